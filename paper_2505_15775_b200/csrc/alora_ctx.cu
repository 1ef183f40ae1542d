// alora_ctx.cu -- context creation (validation, re-layout of the sparse data, upload) and the
// small non-templated kernels (ordered final reductions, long-constraint finish, low-rank term).
#include <algorithm>
#include <cmath>
#include <cstring>
#include <numeric>

#include "alora_internal.h"
#include "rows_tiled.cuh"

namespace alora {

alora_status fail(alora_ctx* c, alora_status s, const std::string& msg) {
  if (c) c->err = msg;
  return s;
}

// ---------------------------------------------------------------------------------------------
// small kernels
// ---------------------------------------------------------------------------------------------
// one block per long constraint: ordered sum of its chunk partials, then the per-constraint finish.
__global__ void k_long_finish(int mode, int64_t m, const int* long_cons, const int64_t* long_chptr,
                              const double* ch_out, const double* y, const double* b, double sigma,
                              double* z, double* lam, double* partials, const FinArgs fin) {
  __shared__ double sm[3][kBlock / 32];
  ALORA_GRID_DEP();
  const int slot = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int64_t c0 = long_chptr[slot], c1 = long_chptr[slot + 1];
  double v[3] = {0.0, 0.0, 0.0};
  for (int64_t c = c0 + threadIdx.x; c < c1; c += kBlock) {
    v[0] += ch_out[3 * c]; v[1] += ch_out[3 * c + 1]; v[2] += ch_out[3 * c + 2];
  }
  for (int k = 0; k < 3; ++k) { double t = warp_sum(v[k]); if (lane == 0) sm[k][warp] = t; }
  __syncthreads();
  if (threadIdx.x < kNStat) partials[(int64_t)slot * kNStat + threadIdx.x] = 0.0;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t[3] = {0.0, 0.0, 0.0};
    for (int k = 0; k < 3; ++k) for (int wv = 0; wv < kBlock / 32; ++wv) t[k] += sm[k][wv];
    double st[kNStat];
    for (int s = 0; s < kNStat; ++s) st[s] = 0.0;
    const int64_t i = long_cons[slot];
    if (mode == CONS_EVAL) {
      cons_finish<CONS_EVAL>(st, i, t[0], t[1], t[2], y, b, sigma, z, lam);
    } else {
      cons_finish<CONS_LS>(st, i, t[0], t[1], t[2], y, b, sigma, z, lam);
    }
    for (int s = 0; s < kNStat; ++s) partials[(int64_t)slot * kNStat + s] = st[s];
  }
  finish_partials(fin);
}

// Low-rank cost term: T = U^T X (pC x r).  Per-block partials, then the block that finishes last (ticket) sums
// them in block order: Tm[p][c], and optionally Ts = s_p * Tm.  blockDim.x = r * rpb.
// gridDim.y = 2: two matrices in one launch (the line search: R -> Tm, D -> Tm2), each with its own partial rows and
// its own ticket word.
template <typename T>
__global__ void k_lowrank(const T* X0, const T* X1, int64_t n, int r, int64_t ld, const T* U, int pC, double* part0, const double* s,
                          double* Tm0, double* Tm1, double* Ts, unsigned int* ticket0) {
  extern __shared__ double lsm[];  // [pC][blockDim.x]
  __shared__ unsigned int s_last;
  ALORA_GRID_DEP();
  const T* const X = blockIdx.y ? X1 : X0;
  double* const Tm = blockIdx.y ? Tm1 : Tm0;
  double* const part = part0 + (size_t)blockIdx.y * gridDim.x * pC * r;
  unsigned int* const ticket = ticket0 + blockIdx.y;
  const int c = threadIdx.x % r, slot = threadIdx.x / r, rpb = blockDim.x / r;
  double acc[8];
  for (int p = 0; p < 8; ++p) acc[p] = 0.0;
  for (int64_t row = (int64_t)blockIdx.x * rpb + slot; row < n; row += (int64_t)gridDim.x * rpb) {
    const double xv = (double)X[row * ld + c];
    for (int p = 0; p < pC; ++p) acc[p] += (double)U[row * pC + p] * xv;
  }
  for (int p = 0; p < pC; ++p) lsm[p * blockDim.x + threadIdx.x] = acc[p];
  __syncthreads();
  if (slot == 0) {
    for (int p = 0; p < pC; ++p) {
      double v = 0.0;
      for (int s2 = 0; s2 < rpb; ++s2) v += lsm[p * blockDim.x + s2 * r + c];
      part[((int64_t)blockIdx.x * pC + p) * r + c] = v;
    }
  }
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) s_last = (atomicAdd(ticket, 1u) == gridDim.x - 1) ? 1u : 0u;
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  // thread t sums entry t % pr over the blocks t / pr, t / pr + nsl, ... ; the nsl slices are then added in order
  const int nblk = gridDim.x, pr = pC * r, nsl = max(1, (int)blockDim.x / pr);
  for (int idx0 = 0; idx0 < pr; idx0 += blockDim.x) {   // one pass unless pC * r > blockDim.x
    const int idx = idx0 + (int)threadIdx.x % pr, sl = (int)threadIdx.x / pr;
    double v = 0.0;
    if (sl < nsl && idx < pr) {
      int bk = sl;
      for (; bk + 3 * nsl < nblk; bk += 4 * nsl) {
        const double v0 = __ldcg(part + (int64_t)bk * pr + idx), v1 = __ldcg(part + (int64_t)(bk + nsl) * pr + idx);
        const double v2 = __ldcg(part + (int64_t)(bk + 2 * nsl) * pr + idx), v3 = __ldcg(part + (int64_t)(bk + 3 * nsl) * pr + idx);
        v += v0; v += v1; v += v2; v += v3;
      }
      for (; bk < nblk; bk += nsl) v += __ldcg(part + (int64_t)bk * pr + idx);
    }
    __syncthreads();
    lsm[threadIdx.x] = v;
    __syncthreads();
    if (sl == 0 && idx < pr) {
      double t = 0.0;
      for (int k = 0; k < nsl; ++k) t += lsm[k * pr + (idx - idx0)];
      Tm[idx] = t;
      if (Ts) Ts[idx] = s[idx / r] * t;
    }
  }
  if (threadIdx.x == 0) *ticket = 0u;
}

// lambda = y - sigma (z - b)
__global__ void k_lambda(int64_t m, const double* y, const double* z, const double* b, double sigma, double* lam) {
  ALORA_GRID_DEP();
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < m; i += (int64_t)gridDim.x * blockDim.x)
    lam[i] = y[i] - sigma * (z[i] - b[i]);
}

int pick_vec(const alora_ctx* c, int64_t ld, const void* p0, const void* p1, const void* p2) {
  const int maxv = (int)(16 / c->esz);
  for (int v = maxv; v > 1; v /= 2) {
    const size_t al = (size_t)v * c->esz;
    if (ld % v) continue;
    if (((uintptr_t)p0 % al) || ((uintptr_t)p1 % al) || ((uintptr_t)p2 % al)) continue;
    return v;
  }
  return 1;
}

// mu_dev == NULL in alora_smatvec / alora_lanczos: lambda = y - sigma (z - b) of the last alora_eval.
// The general class wrote it during that evaluation (c->lam); the diagonal class never stores it (it is formed and
// consumed inside the fused pass), so it is recomputed here from that evaluation's z.
alora_status resolve_mu(alora_ctx* c, const double** mu, const char* who) {
  if (*mu || c->m == 0) return ALORA_OK;
  if (!c->have_eval) return fail(c, ALORA_ESTATE, std::string(who) + ": mu_dev == NULL needs a preceding alora_eval");
  if (c->cls == 1) { *mu = c->lam; return ALORA_OK; }
  if (!c->lam_auto) ALORA_CUDA(c, c->pool.alloc((void**)&c->lam_auto, sizeof(double) * c->m));
  const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((c->m + 255) / 256, (int64_t)c->num_sms * 8));
  k_lambda<<<grid, 256, 0, c->stream>>>(c->m, c->y, c->z_last, c->b, c->sigma, c->lam_auto);
  c->launches++;
  ALORA_CUDA(c, cudaGetLastError());
  *mu = c->lam_auto;
  return ALORA_OK;
}

// the scalars of the last evaluation: device-to-host copies into the pinned block (no synchronisation), and their
// assembly into stats[8] once the stream has been synchronised
alora_status stats_enqueue(alora_ctx* c, int r_lowrank) {
  ALORA_CUDA(c, cudaMemcpyAsync(c->pinned, c->stats_dev, sizeof(double) * kNStat, cudaMemcpyDeviceToHost, c->stream));
  if (c->pC && c->cls == 1)
    ALORA_CUDA(c, cudaMemcpyAsync(c->pinned + 64, c->TmR, sizeof(double) * c->pC * r_lowrank, cudaMemcpyDeviceToHost, c->stream));
  return ALORA_OK;
}
void stats_finish(alora_ctx* c, int r_lowrank, double stats[8]) {
  const double* p = c->pinned;
  double cx = p[ES_CX];
  if (c->pC && c->cls == 1)
    for (int q = 0; q < c->pC; ++q) {
      double t = 0.0;
      for (int k = 0; k < r_lowrank; ++k) t += p[64 + q * r_lowrank + k] * p[64 + q * r_lowrank + k];
      cx += c->s_host[q] * t;
    }
  stats[1] = cx; stats[2] = p[ES_YQ]; stats[3] = p[ES_QQ]; stats[4] = p[ES_GG]; stats[5] = p[ES_GR]; stats[6] = p[ES_LZ]; stats[7] = 0.0;
  stats[0] = cx - p[ES_YQ] + 0.5 * c->sigma * p[ES_QQ];
}

}  // namespace alora

// ---------------------------------------------------------------------------------------------
// hot-path calls: alora_eval / alora_linesearch / alora_smatvec
// ---------------------------------------------------------------------------------------------
namespace alora {
namespace {

int vec_slot(int vec) { return vec == 1 ? 0 : vec == 2 ? 1 : 2; }
struct Geo { int vec, nvec, shape, exact; };

// records an event on the ctx stream when kernel timing is on (pairs: before / after the dominant kernel)
void time_mark(alora_ctx* c) {
  if (!c->timing) return;
  // every `timing_every`-th evaluation is bracketed (the two marks of one evaluation share the decision)
  if (c->timing_every > 1 && ((c->timing_calls++ >> 1) % c->timing_every) != 0) return;
  if (c->ev_used == c->ev.size()) {
    if (c->ev.size() >= 16384) return;
    cudaEvent_t e;
    if (cudaEventCreate(&e) != cudaSuccess) return;
    c->ev.push_back(e);
  }
  cudaEventRecord(c->ev[c->ev_used++], c->stream);
}

template <typename T> int grid_rows(alora_ctx* c, int vec, int shape, int mode, int64_t items) {
  int& occ = c->occ_cache[vec_slot(vec)][shape][mode];
  if (!occ) occ = std::max(1, occ_rows(T(), vec, shape, mode));
  const int gpb = kBlock / kShapes[shape].gs;
  const int64_t need = (items + gpb - 1) / gpb;
  return (int)std::max<int64_t>(1, std::min<int64_t>(need, std::min<int64_t>((int64_t)c->num_sms * occ, c->part_cap)));
}
// Row pass of the diagonal class: the tiled kernel on the full tiles plus k_rows on the ragged tail, or
// k_rows alone when the tiled kernel's preconditions do not hold (non-identity diagonal constraints,
// misaligned buffers, tile too large for shared memory).  *nparts = partial rows written.
FinArgs make_fin(const alora_ctx* c, const double* p0, int n0, const double* p1, int n1, const double* p2, int n2, double* out) {
  FinArgs f;
  f.p[0] = p0; f.n[0] = n0; f.p[1] = p1; f.n[1] = n1; f.p[2] = p2; f.n[2] = n2;
  f.out = out; f.ticket = c->ticket;
  return f;
}
FinArgs no_fin() { FinArgs f; f.p[0] = f.p[1] = f.p[2] = nullptr; f.n[0] = f.n[1] = f.n[2] = 0; f.out = nullptr; f.ticket = nullptr; return f; }

template <typename T>
alora_status launch_diag_rows(alora_ctx* c, int vec, int nvec, int exact, int shape, int mode_in, RowArgs<T>& a,
                              const void* dual, double* out) {
  int mode = mode_in;   // ROWS_LS_WARM falls back to ROWS_LS_FUSED when the tiled kernel is not eligible (a.X3 is then cleared)
  const int gs = tiled_shape(mode, shape, c->ell_wide).gs, nit = tiled_shape(mode, shape, c->ell_wide).nit, tr = tile_rows(gs);
  // 1: whole packs, some lanes of a group idle (lane mask); 2: whole packs, all lanes busy.  Rows whose last
  // pack is partially filled (r not a multiple of the vector width) take k_rows.
  const int full = nvec == gs * nit ? 2 : 1;
  const int64_t tiles = c->n / tr;
  bool elig = c->ell_col && exact && tiles > 0 && !((uintptr_t)a.X % 16) && !((uintptr_t)a.X2 % 16) && !((uintptr_t)dual % 16);
  if (mode == ROWS_LS_WARM && (!elig || !a.X3 || ((uintptr_t)a.X3 % 16))) { mode = ROWS_LS_FUSED; a.X3 = nullptr; }   // the warm form exists in the tiled kernel only
  int occ = 0;
  // Share of a row's neighbours that are far (beyond a quarter of L2 in rows of this width): the gathers of such a
  // problem miss L2, their latency is what the pass waits for, and issuing them as predicated load pairs instead of
  // a branch per neighbour pays (config 4: f + grad 1 124 -> 1 039 us, line search 1 283 -> 1 108 us); on a grid,
  // whose neighbours are near, the dense variants are faster with branches (torus, n = 1e6: line search 49.1 -> 47.1
  // us; n = 1.6e7: f + grad 597 -> 522 us), so the dense variants exist in both forms.
  bool sel = c->sel > 0;
  if (c->sel < 0) {
    const int64_t far_rows = std::max<int64_t>(1, (int64_t)(c->l2_bytes / 4) / std::max<int64_t>(1, a.ld * (int64_t)c->esz));
    const int64_t* h = c->ell_hist[(mode == ROWS_LS_FUSED || mode == ROWS_LS_WARM) ? 1 : 0];
    int64_t tot = 0, far = 0;
    for (int b = 0; b < 34; ++b) { tot += h[b]; if (b > 0 && ((int64_t)1 << (b - 1)) >= far_rows) far += h[b]; }
    sel = far * 20 > tot;
  }
  const int flags = (c->ell_wide ? 1 : 0) | (sel ? 2 : 0);
  // L2 policies (RowArgs::l2pol) by size: the single-vector matvec whose streamed slots exceed L2 while its vector
  // fits keeps the vector resident (gathers evict_last, streamed data and output evict_first; config 4: 429 -> 325 us;
  // config 1, all L2-resident: 12.4 -> 14.8 us, so not there); f + grad and line search: no effect measured
  if (c->l2pol < 0)
    a.l2pol = (mode == ROWS_ADJ && (size_t)c->n * (size_t)(ell_slots(c->ell_wide) * (4 + c->esz)) > c->l2_bytes &&
               (size_t)c->n * (size_t)a.ld * c->esz * 2 <= c->l2_bytes * 3) ? 13 : 0;
  auto probe = [&]() {
    int& oc = c->occ_cache[vec_slot(vec)][shape][8 + mode];
    int64_t& key = c->occ_ld[vec_slot(vec)][shape][mode];
    const int64_t want = (a.ld * 4 + full) * 2 + (sel ? 1 : 0);
    if (!oc || key != want) { oc = occ_tiled(T(), vec, shape, mode, full, flags, a.ld); key = want; if (!oc) oc = -1; }
    return oc;
  };
  if (elig) {
    occ = probe();
    if (occ <= 0 && mode == ROWS_LS_WARM) { mode = ROWS_LS_FUSED; a.X3 = nullptr; occ = probe(); }   // the three-tile stage does not fit: cold form
    elig = occ > 0;
  }
  if (!elig) {
    const int grid = grid_rows<T>(c, vec, shape, mode, c->n);
    a.row_begin = 0;
    a.fin = make_fin(c, a.partials, grid, nullptr, 0, nullptr, 0, out);
    ALORA_CUDA(c, launch_rows(vec, shape, mode, a, grid, c->stream));
    c->launches++;
    return ALORA_OK;
  }
  // one launch: the full tiles through the staged pipeline, the ragged tail by the last block, the final sum by
  // whichever block finishes last
  const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(tiles, std::min<int64_t>((int64_t)c->num_sms * occ, c->part_cap / 2)));
  a.tiles = tiles;
  a.fin = make_fin(c, a.partials, grid, nullptr, 0, nullptr, 0, out);
  {
    const cudaError_t e = launch_tiled(vec, shape, mode, full, flags, a, grid, c->stream, c->device);
    if (e != cudaSuccess)
      return fail(c, ALORA_ECUDA, std::string("tiled row kernel launch: ") + cudaGetErrorString(e) + " (vec " + std::to_string(vec) +
                  ", shape " + std::to_string(shape) + ", mode " + std::to_string(mode) + ", full " + std::to_string(full) +
                  ", grid " + std::to_string(grid) + ", blocks/SM " + std::to_string(occ) + ", smem " +
                  std::to_string(tiled_smem_bytes(gs, (int)c->esz, a.ld, mode, c->ell_wide)) + ")");
  }
  c->launches++;
  return ALORA_OK;
}
// The cooperative kernels (k_ent_cw, k_rows_cw) pay when a gathered row is more than one pack (otherwise a thread per
// item already makes one request per row) and the rows do not sit in L1 (measured, profiles/r2b_README.md: config 3
// 466 -> 352 us per step, config 2 adjoint 39 -> 28 us; config 5, n r = 120 KB: 84 -> 96 us).  ALORA_CW=0 / 2: never / always.
inline bool use_cw(const alora_ctx* c, const Geo& g, int r, int64_t ld) {
  if (c->cw == 0 || g.nvec > 32 || (uint64_t)c->n * (uint64_t)ld >= ((uint64_t)1 << 32)) return false;   // 32-bit element offsets
  if (c->cw == 2) return true;
  return g.nvec >= 2 && (size_t)c->n * (size_t)r * c->esz >= ((size_t)1 << 20);
}
// general-class adjoint pass: a group per row; single vectors (Lanczos matvec) on long rows take a warp per row
// (measured on config 3, 60 entries per row: the warp-per-row kernel wins for p = 1, 66 vs 77 us, and loses for
// r = 10, 168 vs 128 us); rows with ~100 entries or more (matrix completion) always take a warp per row
template <typename T> alora_status launch_adj_general(alora_ctx* c, const Geo& g, RowArgs<T>& a, double* out) {
  if (c->nseg > 0) {   // heavy rows: their C part is summed per segment first
    const size_t need = (size_t)c->nseg * (size_t)(g.nvec * g.vec) * c->esz;
    if (need > c->seg_out_bytes) {
      if (c->seg_out) c->pool.release(c->seg_out);
      ALORA_CUDA(c, c->pool.alloc(&c->seg_out, need));
      c->seg_out_bytes = need;
    }
    a.seg_out = (T*)c->seg_out;
    a.nseg = c->nseg;
    const int gs = (int)std::min<int64_t>((c->nseg + kBlock / 32 - 1) / (kBlock / 32), (int64_t)c->num_sms * 8);
    ALORA_CUDA(c, launch_rows_seg(g.vec, g.shape, a, gs, c->stream));
    // second level: a warp per heavy row adds its segments' results into the first segment's slot
    const int gh = (int)std::min<int64_t>((c->nheavy + kBlock / 32 - 1) / (kBlock / 32), (int64_t)c->num_sms * 8);
    ALORA_CUDA(c, launch_k(a.pdl != 0, k_heavy_sum<T>, dim3(std::max(1, gh)), dim3(kBlock), 0, c->stream, c->nheavy, (const int*)c->heavy_segptr,
                           (T*)c->seg_out, c->seg_cx, g.nvec * g.vec));
    c->launches += 2;
  }
  if (use_cw(c, g, a.r, a.ld) && !c->row_perm && !c->ep_wide) {
    // cooperative warp per row (k_rows_cw): coalesced entry metadata, one request per gathered row; not for skewed row
    // lengths (config 7: 769 against 474 us) nor for very long rows of thin vectors (k_rows_ep is as fast there)
    int pl2 = 0; while ((1 << pl2) < g.nvec) ++pl2;
    int& occ = c->occ_cw[vec_slot(g.vec)][pl2];
    if (!occ) occ = std::max(1, occ_rows_cw(T(), g.vec, g.nvec));
    const int64_t need = (c->n + kBlock / 32 - 1) / (kBlock / 32);
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(need, std::min<int64_t>((int64_t)c->num_sms * occ, c->part_cap)));
    a.perm = c->row_perm;
    a.fin = make_fin(c, a.fin.p[0], grid, a.fin.p[1], a.fin.n[1], a.fin.p[2], a.fin.n[2], out);
    ALORA_CUDA(c, launch_rows_cw(g.vec, a, grid, c->stream));
  } else if ((c->ep && g.nvec == 1 && !c->row_perm) || c->ep_wide) {
    // very long rows of thin vectors (matrix completion, r <= 8 packs): every lane owns whole rows, 32 entry lanes
    const int eshape = (c->ep_wide && g.nvec > 1 && g.nvec <= 4) ? 7 : (c->ep_wide && g.nvec > 4 && g.nvec <= 8) ? 8 : g.shape;
    int& occ = c->occ_cache[vec_slot(g.vec)][eshape == g.shape ? g.shape : eshape - 7][eshape == g.shape ? 11 : 7];
    if (!occ) occ = std::max(1, occ_rows_ep(T(), g.vec, eshape));
    const int64_t need = (c->n + kBlock / 32 - 1) / (kBlock / 32);
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(need, std::min<int64_t>((int64_t)c->num_sms * occ, c->part_cap)));
    a.fin = make_fin(c, a.fin.p[0], grid, a.fin.p[1], a.fin.n[1], a.fin.p[2], a.fin.n[2], out);
    ALORA_CUDA(c, launch_rows_ep(g.vec, eshape, a, grid, c->stream));
  } else {
    const int grid = grid_rows<T>(c, g.vec, g.shape, ROWS_ADJ, c->n);
    a.perm = c->row_perm;
    a.fin = make_fin(c, a.fin.p[0], grid, a.fin.p[1], a.fin.n[1], a.fin.p[2], a.fin.n[2], out);
    ALORA_CUDA(c, launch_rows(g.vec, g.shape, ROWS_ADJ, a, grid, c->stream));
  }
  c->launches++;
  return ALORA_OK;
}
template <typename T> int grid_cons(alora_ctx* c, int vec, int shape, int mode, int chunked, int64_t items) {
  int& occ = c->occ_cache[vec_slot(vec)][shape][3 + mode * 2 + chunked];
  if (!occ) occ = std::max(1, occ_cons(T(), vec, shape, mode, chunked));
  const int gpb = kBlock / kShapes[shape].gs;
  const int64_t need = (items + gpb - 1) / gpb;
  return (int)std::max<int64_t>(1, std::min<int64_t>(need, std::min<int64_t>((int64_t)c->num_sms * occ, c->part_cap)));
}

alora_status geometry(alora_ctx* c, int32_t r, int64_t ld, const void* p0, const void* p1, const void* p2, Geo& g) {
  if (r < 1 || ld < r) return fail(c, ALORA_EINVAL, "need 1 <= r <= ld");
  if (((uintptr_t)p0 % c->esz) || ((uintptr_t)p1 % c->esz) || ((uintptr_t)p2 % c->esz)) return fail(c, ALORA_EINVAL, "misaligned pointer");
  g.vec = pick_vec(c, ld, p0, p1, p2);
  // padded rows (ld > r) on the staged-tile path: a narrower pack that divides r keeps that path eligible
  if (c->cls == 0 && c->ell_col) while (g.vec > 1 && r % g.vec) g.vec /= 2;
  g.nvec = (r + g.vec - 1) / g.vec;
  g.shape = shape_index(g.nvec);
  g.exact = (g.nvec * g.vec == r);
  if (g.shape < 0) return fail(c, ALORA_EINVAL, "r too large for this alignment (<= 64 packs per row)");
  return ALORA_OK;
}

// Programmatic dependent launch (launch_k, ALORA_GRID_DEP): the blocks of the next kernel are scheduled and run their
// prologue while the current one drains.  Measured per step: config 0 32.9 -> 28.0 us, config 1 96.3 -> 93.0 us, config 2
// 154.7 -> 132.7 us (11 launches), config 5 79.9 -> 75.2 us, config 6 134.6 -> 131.9 us, config 3 324 -> 319 us; SLOWER at
// n = 2^24 (2 498 -> 2 528 us) and on the skewed rows of config 7 (953 -> 970 us), hence the two conditions.
inline bool use_pdl(const alora_ctx* c, int64_t ld) {
  return c->pdl == 2 || (c->pdl == 1 && !c->row_perm && (size_t)c->n * (size_t)ld * c->esz <= 4 * c->l2_bytes);
}
template <typename T> void fill_rows(alora_ctx* c, RowArgs<T>& a, const Geo& g, const T* X, int r, int64_t ld) {
  a.n = c->n; a.r = r; a.ld = ld; a.nvec = g.nvec; a.exact = g.exact; a.X = X; a.X2 = nullptr; a.X3 = nullptr; a.Out = nullptr;
  a.perm = nullptr; a.l2pol = c->l2pol < 0 ? 0 : c->l2pol;
  a.pdl = use_pdl(c, ld);
  a.c_rowptr = c->c_rowptr; a.c_col = c->c_col; a.c_val = (const T*)c->c_val; a.dC = (const T*)c->dC;
  a.dcons = c->dcons; a.da = (const T*)c->da;
  a.a_rowptr = c->a_rowptr; a.a_col = c->a_col; a.a_val = (const T*)c->a_val; a.a_cons = c->a_cons;
  a.y = c->y; a.b = c->b; a.sigma = c->sigma; a.w = nullptr; a.z = nullptr;
  a.pC = 0; a.U = (const T*)c->U; a.Ts = c->Ts; a.scale = 1.0; a.diag_class = (c->cls == 0);
  a.partials = c->part_rows; a.row_begin = 0; a.tiles = 0;
  a.ell_col = c->ell_col; a.ell_val = (const T*)c->ell_val;
  a.nseg = 0; a.nheavy = c->nheavy; a.seg_row = c->seg_row; a.seg_beg = c->seg_beg; a.seg_end = c->seg_end;
  a.heavy_rows = c->heavy_rows; a.heavy_segptr = c->heavy_segptr; a.seg_out = (T*)c->seg_out; a.seg_cx = c->seg_cx;
  a.fin = no_fin();
}
template <typename T> void fill_cons(alora_ctx* c, ConsArgs<T>& a, const Geo& g, const T* X, const T* X2, int r, int64_t ld) {
  a.n = c->n; a.r = r; a.ld = ld; a.nvec = g.nvec; a.exact = g.exact; a.X = X; a.X2 = X2; a.m = c->m;
  a.ptr = c->f_ptr; a.e_row = c->f_row; a.e_col = c->f_col; a.e_val = (const T*)c->f_val;
  a.y = c->y; a.b = c->b; a.sigma = c->sigma; a.z = nullptr; a.lam = c->lam;
  a.nchunk = 0; a.ch_beg = c->ch_beg; a.ch_end = c->ch_end; a.ch_out = c->ch_out; a.partials = c->part_cons;
  a.nchunk_A = c->nchunk_A; a.part_chunk = c->part_chunk;
  a.fin = no_fin(); a.pdl = use_pdl(c, ld);
}

// T = U^T X (pC x r) into Tm, optionally Ts = s * Tm
template <typename T> alora_status lowrank(alora_ctx* c, const T* X, int r, int64_t ld, double* Tm, bool want_Ts,
                                           const T* X2 = nullptr, double* Tm2 = nullptr) {
  if (r > c->lr_rmax) return fail(c, ALORA_EINVAL, "low-rank cost term supports r <= 256");
  // Large blocks (up to 1024 threads, shared memory pC * threads doubles <= 48 KB) and a grid of about 8 rows per thread:
  // both phases of the kernel are latency chains (the row loop, then the last block's ordered sum over the blocks), and
  // this keeps both short (config 2, n = 20 000, r = 24: 296 blocks of 240 threads took 14 us, 78 blocks of 768 take 11 under ncu).
  const int tmax = std::min(1024, 6144 / std::max(1, c->pC));
  const int rpb = std::max(1, std::min(32, tmax / r)), threads = r * rpb;   // <= 32 row slots: their sums are added by one thread per column
  const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(c->lr_grid, (c->n + (int64_t)rpb * 8 - 1) / ((int64_t)rpb * 8)));
  ALORA_CUDA(c, launch_k(use_pdl(c, ld), k_lowrank<T>, dim3(grid, X2 ? 2 : 1), dim3(threads), sizeof(double) * c->pC * threads, c->stream,
                         X, X2, c->n, r, ld, (const T*)c->U, c->pC, c->lr_part, (const double*)c->s_dev, Tm, Tm2,
                         want_Ts ? c->Ts : (double*)nullptr, c->lr_ticket));
  c->launches++;
  ALORA_CUDA(c, cudaGetLastError());
  return ALORA_OK;
}

// Forward pass of the general class with the cooperative entry kernel: k_ent_cw over the entries, then (unless every
// constraint is a single entry) k_cons_fin per short constraint and k_long_fin_e per long one.  `nent` entries are
// walked (the constraint entries; for the line search C's sym-upper list as well).  The partial rows land in
// part_cons (*ge rows), part_chunk (*gf rows) and part_long (nlong_A rows); `last_fin`, if given, is attached to the
// last kernel launched (the line search ends here; an evaluation ends with the adjoint pass).
template <typename T>
alora_status forward_cw(alora_ctx* c, const Geo& g, int mode, ConsArgs<T>& ca, int64_t nent, int* ge, int* gf, double* last_out) {
  const int K = 3;
  const size_t need = (size_t)std::max<int64_t>(1, c->nf_A) * K * c->esz;
  if (!c->e_out) ALORA_CUDA(c, c->pool.alloc(&c->e_out, need));
  ca.nent = nent; ca.nf_A = c->nf_A; ca.e_out = (T*)c->e_out; ca.long_cons = c->long_cons;
  ca.npc = c->uniform_npc;
  const bool single = c->single_entry, fin_k = !single && c->uniform_npc <= 1 && c->m > 0, longs = fin_k && c->nlong_A > 0;
  *ge = (int)std::max<int64_t>(1, std::min<int64_t>((nent + kBlock - 1) / kBlock, std::min<int64_t>((int64_t)c->num_sms * 8, c->part_cap)));
  *gf = fin_k ? (int)std::max<int64_t>(1, std::min<int64_t>((c->m + kBlock - 1) / kBlock, std::min<int64_t>((int64_t)c->num_sms * 8, c->part_cap))) : 0;
  auto fin_all = [&]() { return make_fin(c, c->part_cons, *ge, c->part_chunk, *gf, c->part_long, longs ? c->nlong_A : 0, last_out); };
  ca.partials = c->part_cons; ca.part_chunk = c->part_chunk;
  ca.fin = (last_out && !fin_k) ? fin_all() : no_fin();
  ALORA_CUDA(c, launch_ent_cw(g.vec, mode, single ? 1 : 0, ca, *ge, c->stream));
  c->launches++;
  if (fin_k) {
    ca.fin = (last_out && !longs) ? fin_all() : no_fin();
    if (mode == CONS_EVAL) ALORA_CUDA(c, launch_k(ca.pdl, k_cons_fin<T, CONS_EVAL>, dim3(*gf), dim3(kBlock), 0, c->stream, ca));
    else ALORA_CUDA(c, launch_k(ca.pdl, k_cons_fin<T, CONS_LS>, dim3(*gf), dim3(kBlock), 0, c->stream, ca));
    c->launches++;
    if (longs) {
      ca.fin = last_out ? fin_all() : no_fin();
      if (mode == CONS_EVAL) ALORA_CUDA(c, launch_k(ca.pdl, k_long_fin_e<T, CONS_EVAL>, dim3(c->nlong_A), dim3(kLongFinThreads), 0, c->stream, ca, c->part_long));
      else ALORA_CUDA(c, launch_k(ca.pdl, k_long_fin_e<T, CONS_LS>, dim3(c->nlong_A), dim3(kLongFinThreads), 0, c->stream, ca, c->part_long));
      c->launches++;
    }
  }
  ca.fin = no_fin();
  ALORA_CUDA(c, cudaGetLastError());
  return ALORA_OK;
}

template <typename T> alora_status eval_impl(alora_ctx* c, const T* R, int32_t r, int64_t ld, T* G, double* z_dev) {
  Geo g;
  alora_status s = geometry(c, r, ld, R, G, nullptr, g);
  if (s != ALORA_OK) return s;
  if (G && (const void*)G == (const void*)R) return fail(c, ALORA_EINVAL, "G must not alias R");
  double* zout = z_dev ? z_dev : c->z_int;
  RowArgs<T> a;
  fill_rows(c, a, g, R, r, ld);
  a.Out = G; a.scale = 2.0;
  if (c->cls == 0) {
    a.z = zout;
    time_mark(c);
    s = launch_diag_rows<T>(c, g.vec, g.nvec, g.exact, g.shape, ROWS_FUSED_EVAL, a, c->y, c->stats_dev);
    if (s != ALORA_OK) return s;
    time_mark(c);
  } else {
    if (c->pC) { s = lowrank<T>(c, R, r, ld, c->TmR, true); if (s != ALORA_OK) return s; a.pC = c->pC; }
    ConsArgs<T> ca;
    fill_cons(c, ca, g, R, (const T*)nullptr, r, ld);
    ca.z = zout;
    int gc = 0;
    if (use_cw(c, g, r, ld) && c->m > 0) {
      int ge = 0, gf = 0;
      s = forward_cw<T>(c, g, CONS_EVAL, ca, c->nf_A, &ge, &gf, nullptr);
      if (s != ALORA_OK) return s;
      a.w = c->lam; a.diag_class = 0;
      const bool fin_k = !c->single_entry && c->uniform_npc <= 1;
      a.fin = make_fin(c, c->part_rows, 0, fin_k ? c->part_chunk : c->part_cons, fin_k ? gf : ge, c->part_long,
                       (fin_k && c->nlong_A > 0) ? c->nlong_A : 0, nullptr);   // last kernel of the call
      time_mark(c);
      s = launch_adj_general<T>(c, g, a, c->stats_dev);
      if (s != ALORA_OK) return s;
      time_mark(c);
      ALORA_CUDA(c, cudaGetLastError());
      c->z_last = zout; c->have_eval = true;
      return ALORA_OK;
    }
    if (c->m > 0) {
      if (c->single_entry || c->short_cons) {
        gc = (int)std::min<int64_t>((c->m + kBlock - 1) / kBlock, std::min<int64_t>((int64_t)c->num_sms * 8, c->part_cap));
        ALORA_CUDA(c, launch_cons1(g.vec, CONS_EVAL, c->single_entry ? 1 : 0, ca, gc, c->stream));
      } else {
        gc = grid_cons<T>(c, g.vec, g.shape, CONS_EVAL, 0, c->m);
        ALORA_CUDA(c, launch_cons(g.vec, g.shape, CONS_EVAL, 0, ca, gc, c->stream));
      }
      c->launches++;
    }
    if (c->nchunk_A > 0) {
      ca.nchunk = c->nchunk_A;
      const int gk = grid_cons<T>(c, g.vec, g.shape, CONS_EVAL, 1, c->nchunk_A);
      ALORA_CUDA(c, launch_cons(g.vec, g.shape, CONS_EVAL, 1, ca, gk, c->stream));
      k_long_finish<<<c->nlong_A, kBlock, 0, c->stream>>>(CONS_EVAL, c->m, c->long_cons, c->long_chptr, c->ch_out, c->y,
                                                         c->b, c->sigma, zout, c->lam, c->part_long, no_fin());
      c->launches += 2;
    }
    a.w = c->lam; a.diag_class = 0;
    a.fin = make_fin(c, c->part_rows, 0, c->part_cons, gc, c->part_long, c->nlong_A, nullptr);   // last kernel of the call
    time_mark(c);
    s = launch_adj_general<T>(c, g, a, c->stats_dev);
    if (s != ALORA_OK) return s;
    time_mark(c);
  }
  ALORA_CUDA(c, cudaGetLastError());
  c->z_last = zout; c->have_eval = true;
  return ALORA_OK;
}

alora_status fetch_stats(alora_ctx* c, int r_lowrank, double stats[8]) {
  alora_status s = stats_enqueue(c, r_lowrank);
  if (s != ALORA_OK) return s;
  ALORA_CUDA(c, cudaStreamSynchronize(c->stream));
  stats_finish(c, r_lowrank, stats);
  return ALORA_OK;
}

template <typename T> alora_status ls_impl(alora_ctx* c, const T* R, const T* D, int32_t r, int64_t ld, const T* G_warm) {
  Geo g;
  alora_status s = geometry(c, r, ld, R, D, nullptr, g);
  if (s != ALORA_OK) return s;
  if (c->cls == 0) {
    RowArgs<T> a;
    fill_rows(c, a, g, R, r, ld);
    a.X2 = D; a.X3 = G_warm;
    a.ell_col = c->ellu_col; a.ell_val = (const T*)c->ellu_val;
    s = launch_diag_rows<T>(c, g.vec, g.nvec, g.exact, g.shape, G_warm ? ROWS_LS_WARM : ROWS_LS_FUSED, a, c->y, c->ls_dev);
    if (s != ALORA_OK) return s;
    c->ls_used_g = a.X3 != nullptr;   // launch_diag_rows drops it when the tiled kernel is not eligible
  } else {
    if (c->pC) {
      s = lowrank<T>(c, R, r, ld, c->TmR, false, D, c->TmD); if (s != ALORA_OK) return s;   // both in one launch
    }
    ConsArgs<T> ca;
    fill_cons(c, ca, g, R, D, r, ld);
    if (use_cw(c, g, r, ld) && c->nf_A + c->nf_C > 0) {
      int ge = 0, gf = 0;
      s = forward_cw<T>(c, g, CONS_LS, ca, c->nf_A + c->nf_C, &ge, &gf, c->ls_dev);
      if (s != ALORA_OK) return s;
      c->have_ls = true;
      return ALORA_OK;
    }
    // launches: k_cons (short constraints), k_cons_chunk (chunks of long constraints and of C's list),
    // k_long_finish (long constraints); whichever comes last also does the final sum
    const bool chunks = c->nchunk_all > 0, longs = c->nlong_A > 0;
    int gc = 0, gk = 0;
    if (chunks) gk = grid_cons<T>(c, g.vec, g.shape, CONS_LS, 1, c->nchunk_all);
    if (c->m > 0) {
      gc = (c->single_entry || c->short_cons) ? (int)std::min<int64_t>((c->m + kBlock - 1) / kBlock, std::min<int64_t>((int64_t)c->num_sms * 8, c->part_cap))
                           : grid_cons<T>(c, g.vec, g.shape, CONS_LS, 0, c->m);
      if (!chunks) ca.fin = make_fin(c, c->part_cons, gc, nullptr, 0, nullptr, 0, c->ls_dev);
      if (c->single_entry || c->short_cons) ALORA_CUDA(c, launch_cons1(g.vec, CONS_LS, c->single_entry ? 1 : 0, ca, gc, c->stream));
      else ALORA_CUDA(c, launch_cons(g.vec, g.shape, CONS_LS, 0, ca, gc, c->stream));
      ca.fin = no_fin();
      c->launches++;
    }
    if (chunks) {
      ca.nchunk = c->nchunk_all;
      if (!longs) ca.fin = make_fin(c, c->part_cons, gc, c->part_chunk, gk, nullptr, 0, c->ls_dev);
      ALORA_CUDA(c, launch_cons(g.vec, g.shape, CONS_LS, 1, ca, gk, c->stream));
      c->launches++;
      if (longs) {
        k_long_finish<<<c->nlong_A, kBlock, 0, c->stream>>>(CONS_LS, c->m, c->long_cons, c->long_chptr, c->ch_out, c->y,
                                                          c->b, c->sigma, nullptr, nullptr, c->part_long,
                                                          make_fin(c, c->part_cons, gc, c->part_chunk, gk, c->part_long, c->nlong_A, c->ls_dev));
        c->launches++;
      }
    } else if (c->m == 0) {
      ALORA_CUDA(c, cudaMemsetAsync(c->ls_dev, 0, sizeof(double) * kNStat, c->stream));
    }
  }
  ALORA_CUDA(c, cudaGetLastError());
  c->have_ls = true;
  return ALORA_OK;
}


alora_status fetch_ls(alora_ctx* c, int r, double p[5]) {
  ALORA_CUDA(c, cudaMemcpyAsync(c->pinned, c->ls_dev, sizeof(double) * kNStat, cudaMemcpyDeviceToHost, c->stream));
  if (c->ls_warm) ALORA_CUDA(c, cudaMemcpyAsync(c->pinned + 16, c->ls_warm_stats, sizeof(double) * kNStat, cudaMemcpyDeviceToHost, c->stream));
  const bool lr = c->pC && c->cls == 1;
  if (lr) {
    ALORA_CUDA(c, cudaMemcpyAsync(c->pinned + 64, c->TmR, sizeof(double) * c->pC * r, cudaMemcpyDeviceToHost, c->stream));
    ALORA_CUDA(c, cudaMemcpyAsync(c->pinned + 64 + 8 * 256, c->TmD, sizeof(double) * c->pC * r, cudaMemcpyDeviceToHost, c->stream));
  }
  ALORA_CUDA(c, cudaStreamSynchronize(c->stream));
  const double* s = c->pinned;
  double cRR = s[LS_CRR], cRD = s[LS_CRD], cDD = s[LS_CDD];
  if (lr)
    for (int q = 0; q < c->pC; ++q) {
      const double* tr = s + 64 + q * r; const double* td = s + 64 + 8 * 256 + q * r;
      double rr = 0, rd = 0, dd = 0;
      for (int k = 0; k < r; ++k) { rr += tr[k] * tr[k]; rd += tr[k] * td[k]; dd += td[k] * td[k]; }
      cRR += c->s_host[q] * rr; cRD += c->s_host[q] * rd; cDD += c->s_host[q] * dd;
    }
  const double sg = c->sigma;
  p[0] = cRR - s[LS_YQ] + 0.5 * sg * s[LS_QQ];
  if (c->ls_warm) {   // p0 = f(R) of the evaluation the caller vouched for (its <C,RR^T> already holds the low-rank term)
    const double* e = c->pinned + 16;
    double cx = e[ES_CX];
    if (lr) for (int q = 0; q < c->pC; ++q) { const double* tr = s + 64 + q * r; double rr = 0; for (int k = 0; k < r; ++k) rr += tr[k] * tr[k]; cx += c->s_host[q] * rr; }
    p[0] = cx - e[ES_YQ] + 0.5 * sg * e[ES_QQ];
  }
  p[1] = c->ls_used_g ? s[LS_CRD]   // warm form with the evaluation's gradient: the slot carries <G,D> = d/d alpha f(R + alpha D) at 0
                      : 2.0 * cRD - s[LS_YQ1] + sg * s[LS_QQ1];
  p[2] = cDD - s[LS_YQ2] + 0.5 * sg * s[LS_Q11] + sg * s[LS_QQ2];
  p[3] = sg * s[LS_Q12];
  p[4] = 0.5 * sg * s[LS_Q22];
  return ALORA_OK;
}

template <typename T> alora_status matvec_impl(alora_ctx* c, const double* mu, const T* V, int32_t p, T* W) {
  Geo g;
  alora_status s = geometry(c, p, p, V, W, nullptr, g);
  if (s != ALORA_OK) return s;
  RowArgs<T> a;
  fill_rows(c, a, g, V, p, p);
  a.Out = W; a.scale = 1.0; a.w = mu; a.diag_class = (c->cls == 0);
  if (c->pC) { s = lowrank<T>(c, V, p, p, c->TmD, true); if (s != ALORA_OK) return s; a.pC = c->pC; }
  if (c->cls == 0) {
    s = launch_diag_rows<T>(c, g.vec, g.nvec, g.exact, g.shape, ROWS_ADJ, a, mu, c->mv_dev);
    if (s != ALORA_OK) return s;
  } else {
    a.fin = make_fin(c, c->part_rows, 0, nullptr, 0, nullptr, 0, nullptr);
    s = launch_adj_general<T>(c, g, a, c->mv_dev);
    if (s != ALORA_OK) return s;
  }
  ALORA_CUDA(c, cudaGetLastError());
  return ALORA_OK;
}


}  // namespace
}  // namespace alora

using namespace alora;

extern "C" alora_status alora_eval(alora_ctx* c, const void* R, int32_t r, int64_t ld, void* G, double* z_dev, double stats[8]) {
  if (!c || !R) return c ? fail(c, ALORA_EINVAL, "alora_eval: NULL argument") : ALORA_EINVAL;
  if (!c->have_dual) return fail(c, ALORA_ESTATE, "alora_eval before alora_set_dual");
  ALORA_CUDA(c, cudaSetDevice(c->device));
  alora_status s = c->dtype == ALORA_F32 ? eval_impl<float>(c, (const float*)R, r, ld, (float*)G, z_dev)
                                         : eval_impl<double>(c, (const double*)R, r, ld, (double*)G, z_dev);
  if (s != ALORA_OK) return s;
  c->last_eval_r = r; c->last_eval_R = R; c->last_eval_ld = ld; c->last_eval_G = G;
  return stats ? fetch_stats(c, r, stats) : ALORA_OK;
}

extern "C" alora_status alora_get_stats(alora_ctx* c, double stats[8]) {
  if (!c || !stats) return ALORA_EINVAL;
  if (!c->have_eval) return fail(c, ALORA_ESTATE, "alora_get_stats before alora_eval");
  return fetch_stats(c, c->last_eval_r, stats);
}

extern "C" alora_status alora_get_lambda(alora_ctx* c, double* lam_dev) {
  if (!c) return ALORA_EINVAL;
  if (!lam_dev && c->m > 0) return fail(c, ALORA_EINVAL, "alora_get_lambda: lam_dev is NULL");
  if (!c->have_eval) return fail(c, ALORA_ESTATE, "alora_get_lambda before alora_eval");
  if (c->m == 0) return ALORA_OK;
  const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((c->m + 255) / 256, (int64_t)c->num_sms * 8));
  k_lambda<<<grid, 256, 0, c->stream>>>(c->m, c->y, c->z_last, c->b, c->sigma, lam_dev);
  c->launches++;
  ALORA_CUDA(c, cudaGetLastError());
  return ALORA_OK;
}

extern "C" alora_status alora_eval_host(alora_ctx* c, const void* R_host, int32_t r, int64_t ld, void* G_host, double* z_host,
                                        double stats[8]) {
  if (!c || !R_host || !stats) return c ? fail(c, ALORA_EINVAL, "alora_eval_host: NULL argument") : ALORA_EINVAL;
  if (r < 1 || ld < r) return fail(c, ALORA_EINVAL, "need 1 <= r <= ld");
  ALORA_CUDA(c, cudaSetDevice(c->device));
  const size_t nb = (size_t)c->n * (size_t)ld * c->esz;
  if (nb > c->stage_bytes) {
    if (c->stageR) { c->pool.release(c->stageR); c->pool.release(c->stageG); }
    ALORA_CUDA(c, c->pool.alloc(&c->stageR, nb));
    ALORA_CUDA(c, c->pool.alloc(&c->stageG, nb));
    c->stage_bytes = nb;
  }
  ALORA_CUDA(c, cudaMemcpyAsync(c->stageR, R_host, nb, cudaMemcpyHostToDevice, c->stream));
  alora_status s = alora_eval(c, c->stageR, r, ld, G_host ? c->stageG : nullptr, nullptr, nullptr);
  if (s != ALORA_OK) return s;
  if (G_host) ALORA_CUDA(c, cudaMemcpyAsync(G_host, c->stageG, nb, cudaMemcpyDeviceToHost, c->stream));
  if (z_host) ALORA_CUDA(c, cudaMemcpyAsync(z_host, c->z_int, sizeof(double) * c->m, cudaMemcpyDeviceToHost, c->stream));
  return fetch_stats(c, r, stats);
}

extern "C" alora_status alora_step_host(alora_ctx* c, const void* R_host, const void* D_host, const void* V_host, int32_t r,
                                        int64_t ld, void* G_host, double* z_host, void* W_host, double stats[8], double p[5],
                                        double* vw) {
  if (!c || !R_host || !D_host || !V_host || !stats || !p || !vw) return c ? fail(c, ALORA_EINVAL, "alora_step_host: NULL argument") : ALORA_EINVAL;
  if (r < 1 || ld < r) return fail(c, ALORA_EINVAL, "need 1 <= r <= ld");
  if (!c->have_dual) return fail(c, ALORA_ESTATE, "alora_step_host before alora_set_dual");
  ALORA_CUDA(c, cudaSetDevice(c->device));
  const size_t nb = (size_t)c->n * (size_t)ld * c->esz, nv = (size_t)c->n * c->esz;
  if (nb > c->stage_bytes) {
    if (c->stageR) { c->pool.release(c->stageR); c->pool.release(c->stageG); }
    ALORA_CUDA(c, c->pool.alloc(&c->stageR, nb));
    ALORA_CUDA(c, c->pool.alloc(&c->stageG, nb));
    c->stage_bytes = nb;
  }
  if (nb > c->stage2_bytes) {
    if (c->stageD) { c->pool.release(c->stageD); c->pool.release(c->stageV); c->pool.release(c->stageW); }
    ALORA_CUDA(c, c->pool.alloc(&c->stageD, nb));
    ALORA_CUDA(c, c->pool.alloc(&c->stageV, nv));
    ALORA_CUDA(c, c->pool.alloc(&c->stageW, nv));
    c->stage2_bytes = nb;
  }
  if (!c->stream2) {
    ALORA_CUDA(c, cudaStreamCreateWithFlags(&c->stream2, cudaStreamNonBlocking));
    ALORA_CUDA(c, cudaEventCreateWithFlags(&c->ev_eval, cudaEventDisableTiming));
    ALORA_CUDA(c, cudaEventCreateWithFlags(&c->ev_down, cudaEventDisableTiming));
  }
  // ctx stream: R up, f + grad, D and V up (the host-to-device engine is free again while G comes down), line search,
  // matvec, W down.  stream2: G and z down as soon as f + grad is done.
  ALORA_CUDA(c, cudaMemcpyAsync(c->stageR, R_host, nb, cudaMemcpyHostToDevice, c->stream));
  alora_status s = alora_eval(c, c->stageR, r, ld, G_host ? c->stageG : nullptr, nullptr, nullptr);
  if (s != ALORA_OK) return s;
  ALORA_CUDA(c, cudaEventRecord(c->ev_eval, c->stream));
  ALORA_CUDA(c, cudaStreamWaitEvent(c->stream2, c->ev_eval, 0));
  if (G_host) ALORA_CUDA(c, cudaMemcpyAsync(G_host, c->stageG, nb, cudaMemcpyDeviceToHost, c->stream2));
  if (z_host) ALORA_CUDA(c, cudaMemcpyAsync(z_host, c->z_int, sizeof(double) * c->m, cudaMemcpyDeviceToHost, c->stream2));
  ALORA_CUDA(c, cudaEventRecord(c->ev_down, c->stream2));
  ALORA_CUDA(c, cudaMemcpyAsync(c->stageD, D_host, nb, cudaMemcpyHostToDevice, c->stream));
  ALORA_CUDA(c, cudaMemcpyAsync(c->stageV, V_host, nv, cudaMemcpyHostToDevice, c->stream));
  s = alora_linesearch(c, c->stageR, c->stageD, r, ld, 1, nullptr);
  if (s != ALORA_OK) return s;
  s = alora_smatvec(c, nullptr, c->stageV, 1, c->stageW, nullptr);
  if (s != ALORA_OK) return s;
  if (W_host) ALORA_CUDA(c, cudaMemcpyAsync(W_host, c->stageW, nv, cudaMemcpyDeviceToHost, c->stream));
  ALORA_CUDA(c, cudaMemcpyAsync(c->pinned + 32, c->mv_dev, sizeof(double) * kNStat, cudaMemcpyDeviceToHost, c->stream));
  ALORA_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_down, 0));   // the call's results are complete when the ctx stream is
  s = fetch_stats(c, r, stats);            // synchronises the ctx stream
  if (s != ALORA_OK) return s;
  *vw = c->pinned[32 + ES_GR];
  return fetch_ls(c, r, p);
}

extern "C" alora_status alora_linesearch(alora_ctx* c, const void* R, const void* D, int32_t r, int64_t ld, int32_t warm,
                                         double p[5]) {
  if (!c || !R || !D) return c ? fail(c, ALORA_EINVAL, "alora_linesearch: NULL argument") : ALORA_EINVAL;
  if (!c->have_dual) return fail(c, ALORA_ESTATE, "alora_linesearch before alora_set_dual");
  if (warm && !(c->have_eval && c->last_eval_R == R && c->last_eval_r == r && c->last_eval_ld == ld))
    return fail(c, ALORA_ESTATE, "alora_linesearch(warm): no alora_eval of this R (same pointer, r, ld, dual) is on record");
  ALORA_CUDA(c, cudaSetDevice(c->device));
  c->ls_used_g = false;
  const void* Gw = (warm && c->last_eval_G != D) ? c->last_eval_G : nullptr;   // the gradient of the evaluation on record, if it wrote one
  alora_status s = c->dtype == ALORA_F32 ? ls_impl<float>(c, (const float*)R, (const float*)D, r, ld, (const float*)Gw)
                                         : ls_impl<double>(c, (const double*)R, (const double*)D, r, ld, (const double*)Gw);
  if (s != ALORA_OK) return s;
  c->last_ls_r = r;
  c->ls_warm = warm != 0;
  if (warm) {   // the evaluation's scalars, taken now (a later alora_eval overwrites stats_dev); device-to-device, capturable
    if (!c->ls_warm_stats) ALORA_CUDA(c, c->pool.alloc((void**)&c->ls_warm_stats, sizeof(double) * kNStat));
    ALORA_CUDA(c, cudaMemcpyAsync(c->ls_warm_stats, c->stats_dev, sizeof(double) * kNStat, cudaMemcpyDeviceToDevice, c->stream));
  }
  return p ? fetch_ls(c, r, p) : ALORA_OK;
}

extern "C" alora_status alora_get_linesearch(alora_ctx* c, double p[5]) {
  if (!c || !p) return ALORA_EINVAL;
  if (!c->have_ls) return fail(c, ALORA_ESTATE, "alora_get_linesearch before alora_linesearch");
  return fetch_ls(c, c->last_ls_r, p);
}

extern "C" alora_status alora_smatvec(alora_ctx* c, const double* mu_dev, const void* V, int32_t p, void* W, double* vw) {
  if (!c || !V || !W) return c ? fail(c, ALORA_EINVAL, "alora_smatvec: NULL argument") : ALORA_EINVAL;
  if (V == W) return fail(c, ALORA_EINVAL, "W must not alias V");
  ALORA_CUDA(c, cudaSetDevice(c->device));
  alora_status s = resolve_mu(c, &mu_dev, "alora_smatvec");
  if (s != ALORA_OK) return s;
  s = c->dtype == ALORA_F32 ? matvec_impl<float>(c, mu_dev, (const float*)V, p, (float*)W)
                                         : matvec_impl<double>(c, mu_dev, (const double*)V, p, (double*)W);
  if (s != ALORA_OK) return s;
  if (vw) {
    ALORA_CUDA(c, cudaMemcpyAsync(c->pinned + 32, c->mv_dev, sizeof(double) * kNStat, cudaMemcpyDeviceToHost, c->stream));
    ALORA_CUDA(c, cudaStreamSynchronize(c->stream));
    *vw = c->pinned[32 + ES_GR];
  }
  return ALORA_OK;
}

extern "C" alora_status alora_kernel_timing(alora_ctx* c, int enable) {
  if (!c) return ALORA_EINVAL;
  c->timing = enable != 0; c->timing_every = enable > 1 ? enable : 1; c->timing_calls = 0; c->ev_used = 0;
  return ALORA_OK;
}

extern "C" alora_status alora_kernel_timing_read(alora_ctx* c, double* total_ms, int64_t* count) {
  if (!c || !total_ms || !count) return ALORA_EINVAL;
  ALORA_CUDA(c, cudaStreamSynchronize(c->stream));
  double tot = 0.0; int64_t k = 0;
  for (size_t i = 0; i + 1 < c->ev_used; i += 2) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, c->ev[i], c->ev[i + 1]) == cudaSuccess) { tot += ms; ++k; }
  }
  *total_ms = tot; *count = k; c->ev_used = 0;
  return ALORA_OK;
}
