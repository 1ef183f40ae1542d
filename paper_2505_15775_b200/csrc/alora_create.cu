// alora_create.cu -- alora_create: validation, re-layout of the sparse data (host), upload.
//
// Layouts built here:
//   C          : diagonal dC[n] + off-diagonal full-pattern CSR (c_rowptr, c_col, c_val), columns ascending
//   diag class : per row the id of its single diagonal constraint (dcons) and coefficient (da);
//                both omitted when they are the identity / all ones (MaxCut)
//   general    : row-oriented full pattern of all A_i with constraint ids (a_rowptr, a_col, a_val, a_cons),
//                plus the forward list (f_ptr, f_row, f_col, f_val): coalesced constraint entries followed by
//                C's sym-upper entries, and the chunk tables of the "long" constraints and of C.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>

#include "alora_internal.h"

namespace alora {
namespace {

// every array gets 8 zeroed elements of slack: the bulk copies of rows_tiled.cuh read whole 16-byte
// units and may run up to 3 elements past the logical end
template <typename T> cudaError_t upload(alora_ctx* c, void** dst, const std::vector<T>& v) {
  cudaError_t e = c->pool.alloc(dst, (v.size() + 8) * sizeof(T));
  if (e != cudaSuccess) return e;
  e = cudaMemset(*dst, 0, (v.size() + 8) * sizeof(T));
  if (e == cudaSuccess && !v.empty()) e = cudaMemcpy(*dst, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice);
  return e;
}

struct Ent { int col; double val; int cons; };

// bucket directed entries by row (counting sort), sort each row by (col, cons), merge duplicates
void build_csr(int64_t n, const std::vector<int>& rows, std::vector<Ent>& ents, std::vector<int>& rowptr) {
  std::vector<int64_t> cnt(n + 1, 0);
  for (int rj : rows) cnt[rj + 1]++;
  for (int64_t i = 0; i < n; ++i) cnt[i + 1] += cnt[i];
  std::vector<Ent> out(ents.size());
  {
    std::vector<int64_t> pos(cnt.begin(), cnt.end() - 1);
    for (size_t e = 0; e < ents.size(); ++e) out[pos[rows[e]]++] = ents[e];
  }
  std::vector<Ent> merged;
  merged.reserve(out.size());
  rowptr.assign(n + 1, 0);
  for (int64_t i = 0; i < n; ++i) {
    auto b = out.begin() + cnt[i], e = out.begin() + cnt[i + 1];
    std::sort(b, e, [](const Ent& x, const Ent& y) { return x.col != y.col ? x.col < y.col : x.cons < y.cons; });
    const size_t row_start = merged.size();
    for (auto it = b; it != e; ++it) {
      if (merged.size() > row_start && merged.back().col == it->col && merged.back().cons == it->cons)
        merged.back().val += it->val;
      else
        merged.push_back(*it);
    }
    rowptr[i + 1] = (int)merged.size();
  }
  ents.swap(merged);
}

template <typename T> alora_status build(alora_ctx* c, const alora_problem* P) {
  const int64_t n = P->n, m = P->m;
  // ---- C: diagonal + off-diagonal full pattern --------------------------------------------
  std::vector<double> dC(n, 0.0);
  std::vector<int> rows;
  std::vector<Ent> cents;
  rows.reserve(2 * P->nnzC);
  cents.reserve(2 * P->nnzC);
  for (int64_t e = 0; e < P->nnzC; ++e) {
    const int j = P->C_row[e], k = P->C_col[e];
    const double v = P->C_val[e];
    if (j == k) { dC[j] += v; continue; }
    rows.push_back(j); cents.push_back({k, v, -1});
    rows.push_back(k); cents.push_back({j, v, -1});
  }
  std::vector<int> c_rowptr;
  build_csr(n, rows, cents, c_rowptr);
  if (cents.size() >= (size_t)INT32_MAX) return fail(c, ALORA_EINVAL, "C pattern too large for int32 row pointers");
  c->c_nnz = (int64_t)cents.size();
  {
    std::vector<int> col(cents.size());
    std::vector<T> val(cents.size()), d(n);
    for (size_t e = 0; e < cents.size(); ++e) { col[e] = cents[e].col; val[e] = (T)cents[e].val; }
    for (int64_t j = 0; j < n; ++j) d[j] = (T)dC[j];
    ALORA_CUDA(c, upload(c, (void**)&c->c_rowptr, c_rowptr));
    ALORA_CUDA(c, upload(c, (void**)&c->c_col, col));
    ALORA_CUDA(c, upload(c, &c->c_val, val));
    ALORA_CUDA(c, upload(c, &c->dC, d));
  }
  // ||C||_F (denominator of eq. 77 term 2), low-rank part expanded exactly
  double nc2 = 0.0;
  for (int64_t j = 0; j < n; ++j) nc2 += dC[j] * dC[j];
  for (auto& en : cents) nc2 += en.val * en.val;
  for (int p = 0; p < P->pC; ++p) {
    const double* u = P->C_U + (int64_t)p * n;
    double uCu = 0.0;
    for (int64_t j = 0; j < n; ++j) {
      double t = dC[j] * u[j];
      for (int e = c_rowptr[j]; e < c_rowptr[j + 1]; ++e) t += cents[e].val * u[cents[e].col];
      uCu += u[j] * t;
    }
    nc2 += 2.0 * P->C_s[p] * uCu;
    for (int q = 0; q < P->pC; ++q) {
      const double* v = P->C_U + (int64_t)q * n;
      double uv = 0.0;
      for (int64_t j = 0; j < n; ++j) uv += u[j] * v[j];
      nc2 += P->C_s[p] * P->C_s[q] * uv * uv;
    }
  }
  c->normC = std::sqrt(std::max(0.0, nc2));

  // ---- constraints: coalesce inside each constraint, classify ------------------------------
  std::vector<int64_t> f_ptr(m + 1, 0);
  std::vector<int> f_row, f_col;
  std::vector<double> f_val;
  f_row.reserve(P->nnzA); f_col.reserve(P->nnzA); f_val.reserve(P->nnzA);
  // a single diagonal entry per constraint qualifies for the fused one-pass row kernel -- unless the graph has
  // very heavy rows (power-law degrees): the row kernel gives a row to 1..16 lanes, so a row with tens of thousands
  // of entries would serialise; such problems take the general path, whose adjoint pass is a warp per row and whose
  // line search runs over C's entry list in equal chunks
  int64_t c_maxdeg = 0;
  for (int64_t j = 0; j < n; ++j) c_maxdeg = std::max<int64_t>(c_maxdeg, c_rowptr[j + 1] - c_rowptr[j]);
  bool diag_class = (P->pC == 0) && c_maxdeg <= kGeneralRow;
  std::vector<int> dcons(n, -1);
  std::vector<double> da(n, 0.0);
  {
    std::vector<std::pair<std::pair<int, int>, double>> tmp;
    for (int64_t i = 0; i < m; ++i) {
      tmp.clear();
      for (int64_t e = P->A_ptr[i]; e < P->A_ptr[i + 1]; ++e) tmp.push_back({{P->A_row[e], P->A_col[e]}, P->A_val[e]});
      if (tmp.size() > 1)
        std::sort(tmp.begin(), tmp.end(), [](const auto& x, const auto& y) { return x.first < y.first; });
      const size_t start = f_row.size();
      for (auto& t : tmp) {
        if (f_row.size() > start && f_row.back() == t.first.first && f_col.back() == t.first.second) f_val.back() += t.second;
        else { f_row.push_back(t.first.first); f_col.push_back(t.first.second); f_val.push_back(t.second); }
      }
      f_ptr[i + 1] = (int64_t)f_row.size();
      if (diag_class) {
        if (f_ptr[i + 1] - f_ptr[i] != 1 || f_row.back() != f_col.back() || dcons[f_row.back()] >= 0) diag_class = false;
        else { dcons[f_row.back()] = (int)i; da[f_row.back()] = f_val.back(); }
      }
    }
  }
  c->nf_A = (int64_t)f_row.size();
  c->cls = diag_class ? 0 : 1;
  {
    std::vector<double> bb(P->b, P->b + m);
    ALORA_CUDA(c, upload(c, (void**)&c->b, bb));
    double s = 0.0;
    for (double v : bb) s += v * v;
    c->normb = std::sqrt(s);
  }

  if (diag_class) {
    bool ident = (m == n), ones = true;
    for (int64_t j = 0; j < n; ++j) {
      if (dcons[j] != (int)j) ident = false;
      if (dcons[j] >= 0 && (double)(T)da[j] != 1.0) ones = false;
    }
    if (!ident) ALORA_CUDA(c, upload(c, (void**)&c->dcons, dcons));
    if (!ones) {
      std::vector<T> d(n);
      for (int64_t j = 0; j < n; ++j) d[j] = (T)da[j];
      ALORA_CUDA(c, upload(c, &c->da, d));
    }
    if (ident && ones) {
      // padded ELL blocks for the tiled row kernel: slot u of row j at [j * NU + u]; unused slot = (j, 0)
      int64_t over4 = 0;
      for (int64_t j = 0; j < n; ++j) over4 += (c_rowptr[j + 1] - c_rowptr[j] > 4);
      c->ell_wide = over4 * 10 > n;
      const int kUN = ell_slots(c->ell_wide), kUNL = ell_slots_ls(c->ell_wide);
      std::vector<int> ec((size_t)n * kUN), euc((size_t)n * kUNL);
      std::vector<T> ev((size_t)n * kUN), euv((size_t)n * kUNL);
      // Wide block (meshes): within a row the slots are ordered nearest neighbour first (|col - j| ascending, unused
      // slots last), so that slot u is an in-tile neighbour (read from the staged tile) or a farther one (gathered) for
      // most rows of a warp alike and the kernel's in-tile / gather branch per slot rarely diverges (config 6: f + grad
      // 55.3 -> 53.5 us, line search 63.4 -> 61.6 us).  The narrow block's kernels use predicated load pairs; there the
      // order changes nothing or costs (config 4 line search 1 108 -> 1 140 us), so it keeps the CSR order.
      const char* env_sort = std::getenv("ALORA_ELL_SORT");
      const bool sort_slots = env_sort ? std::atoi(env_sort) != 0 : c->ell_wide;   // pays on the wide block (meshes) only: measured
      auto order_slots = [&](int* col, T* val, int cnt, int64_t j) {
        for (int a = 1; a < cnt; ++a) {   // insertion sort, cnt <= 8
          const int cc = col[a]; const T vv = val[a];
          auto key = [&](int cl, T vl) { return (vl == T(0) && cl == (int)j) ? (int64_t)1 << 40 : std::llabs((long long)cl - (long long)j); };
          int b = a - 1;
          while (b >= 0 && key(col[b], val[b]) > key(cc, vv)) { col[b + 1] = col[b]; val[b + 1] = val[b]; --b; }
          col[b + 1] = cc; val[b + 1] = vv;
        }
      };
      for (int64_t j = 0; j < n; ++j) {
        const int e0 = c_rowptr[j], e1 = c_rowptr[j + 1];
        for (int u = 0; u < kUN; ++u) {
          const int e = e0 + u;
          ec[j * kUN + u] = e < e1 ? cents[e].col : (int)j;
          ev[j * kUN + u] = e < e1 ? (T)cents[e].val : T(0);
        }
        if (sort_slots) order_slots(&ec[j * kUN], &ev[j * kUN], kUN, j);
        if (e1 - e0 > kUN) ec[j * kUN] |= (int)0x80000000;   // more neighbours than slots: walk the CSR tail
        for (int u = 0; u < kUNL; ++u) {   // columns ascend: the upper triangle is the tail of the row's list
          const int e = e1 - kUNL + u;
          const bool up = e >= e0 && cents[e].col > j;
          euc[j * kUNL + u] = up ? cents[e].col : (int)j;
          euv[j * kUNL + u] = up ? (T)cents[e].val : T(0);
        }
        if (sort_slots) order_slots(&euc[j * kUNL], &euv[j * kUNL], kUNL, j);
        if (e1 - kUNL - 1 >= e0 && cents[e1 - kUNL - 1].col > j) euc[j * kUNL] |= (int)0x80000000;
        auto bits = [](int64_t d) { int b = 0; while (d) { ++b; d >>= 1; } return b; };
        for (int u = 0; u < kUN; ++u) { const int cl = ec[j * kUN + u] & 0x7fffffff; if (cl != (int)j) c->ell_hist[0][bits(std::llabs((long long)cl - (long long)j))]++; }
        for (int u = 0; u < kUNL; ++u) { const int cl = euc[j * kUNL + u] & 0x7fffffff; if (cl != (int)j) c->ell_hist[1][bits(std::llabs((long long)cl - (long long)j))]++; }
      }
      ALORA_CUDA(c, upload(c, (void**)&c->ell_col, ec));
      ALORA_CUDA(c, upload(c, &c->ell_val, ev));
      ALORA_CUDA(c, upload(c, (void**)&c->ellu_col, euc));
      ALORA_CUDA(c, upload(c, &c->ellu_val, euv));
    }
  } else {
    // row-oriented full pattern with constraint ids
    rows.clear();
    std::vector<Ent> aents;
    rows.reserve(2 * f_row.size()); aents.reserve(2 * f_row.size());
    for (int64_t i = 0; i < m; ++i)
      for (int64_t e = f_ptr[i]; e < f_ptr[i + 1]; ++e) {
        rows.push_back(f_row[e]); aents.push_back({f_col[e], f_val[e], (int)i});
        if (f_row[e] != f_col[e]) { rows.push_back(f_col[e]); aents.push_back({f_row[e], f_val[e], (int)i}); }
      }
    std::vector<int> a_rowptr;
    build_csr(n, rows, aents, a_rowptr);
    if (aents.size() >= (size_t)INT32_MAX) return fail(c, ALORA_EINVAL, "constraint pattern too large for int32 row pointers");
    c->a_nnz = (int64_t)aents.size();
    c->ep = (c->a_nnz + c->c_nnz) >= 8 * n;
    c->ep_wide = (c->a_nnz + c->c_nnz) >= 96 * n;
    {
      // skewed row lengths (power-law graphs): k_rows walks the rows by decreasing work, so the groups of a warp
      // (and the blocks of a wave) get rows of nearly equal length; counting sort, stable in the row index
      const int64_t mean = (c->a_nnz + c->c_nnz) / std::max<int64_t>(1, n);
      int64_t wmax = 0;
      std::vector<int> work(n);
      for (int64_t j = 0; j < n; ++j) {
        const int cd = c_rowptr[j + 1] - c_rowptr[j];
        const int w = (cd > kHeavyRow ? (cd + kHeavyRow - 1) / kHeavyRow : cd) + (a_rowptr[j + 1] - a_rowptr[j]);
        work[j] = w; wmax = std::max<int64_t>(wmax, w);
      }
      if (!c->ep_wide && wmax > 4 * mean + 16 && !std::getenv("ALORA_NO_ROW_ORDER")) {
        std::vector<int64_t> cnt((size_t)wmax + 2, 0);
        for (int64_t j = 0; j < n; ++j) cnt[(size_t)(wmax - work[j]) + 1]++;
        for (size_t k = 1; k < cnt.size(); ++k) cnt[k] += cnt[k - 1];
        std::vector<int> perm(n);
        for (int64_t j = 0; j < n; ++j) perm[(size_t)cnt[(size_t)(wmax - work[j])]++] = (int)j;
        ALORA_CUDA(c, upload(c, (void**)&c->row_perm, perm));
      }
    }
    if (c_maxdeg > kGeneralRow) {   // power-law graphs: every C row longer than kHeavyRow is segmented
      std::vector<int> seg_row, seg_beg, seg_end, heavy_rows, heavy_segptr(1, 0);
      for (int64_t j = 0; j < n; ++j) {
        const int e0 = c_rowptr[j], e1 = c_rowptr[j + 1];
        if (e1 - e0 <= kHeavyRow) continue;
        for (int e = e0; e < e1; e += kHeavyRow) { seg_row.push_back((int)j); seg_beg.push_back(e); seg_end.push_back(std::min(e + kHeavyRow, e1)); }
        heavy_rows.push_back((int)j); heavy_segptr.push_back((int)seg_row.size());
      }
      c->nseg = (int)seg_row.size(); c->nheavy = (int)heavy_rows.size();
      ALORA_CUDA(c, upload(c, (void**)&c->seg_row, seg_row));
      ALORA_CUDA(c, upload(c, (void**)&c->seg_beg, seg_beg));
      ALORA_CUDA(c, upload(c, (void**)&c->seg_end, seg_end));
      ALORA_CUDA(c, upload(c, (void**)&c->heavy_rows, heavy_rows));
      ALORA_CUDA(c, upload(c, (void**)&c->heavy_segptr, heavy_segptr));
      ALORA_CUDA(c, c->pool.alloc((void**)&c->seg_cx, sizeof(double) * (size_t)c->nseg));
    }
    {
      std::vector<int> col(aents.size()), cons(aents.size());
      std::vector<T> val(aents.size());
      for (size_t e = 0; e < aents.size(); ++e) { col[e] = aents[e].col; val[e] = (T)aents[e].val; cons[e] = aents[e].cons; }
      ALORA_CUDA(c, upload(c, (void**)&c->a_rowptr, a_rowptr));
      ALORA_CUDA(c, upload(c, (void**)&c->a_col, col));
      ALORA_CUDA(c, upload(c, &c->a_val, val));
      ALORA_CUDA(c, upload(c, (void**)&c->a_cons, cons));
    }
    // chunk tables of the long constraints
    std::vector<int64_t> ch_beg, ch_end, long_chptr(1, 0);
    std::vector<int> long_cons;
    for (int64_t i = 0; i < m; ++i) {
      if (f_ptr[i + 1] - f_ptr[i] > kLongThreshold) {
        for (int64_t e = f_ptr[i]; e < f_ptr[i + 1]; e += kChunk) { ch_beg.push_back(e); ch_end.push_back(std::min<int64_t>(e + kChunk, f_ptr[i + 1])); }
        long_cons.push_back((int)i); long_chptr.push_back((int64_t)ch_beg.size());
      }
    }
    c->nchunk_A = (int64_t)ch_beg.size(); c->nlong_A = (int)long_cons.size();
    c->single_entry = m > 0;
    for (int64_t i = 0; i < m && c->single_entry; ++i) c->single_entry = (f_ptr[i + 1] - f_ptr[i] == 1);
    c->short_cons = m > 0 && c->nf_A <= 8 * m;
    if (m > 0 && !c->single_entry) {   // uniform constraints: k_ent_cw finishes them in its own pass
      const int64_t npc = f_ptr[1] - f_ptr[0];
      bool uni = npc > 1 && npc <= 32 && 32 % npc == 0;
      for (int64_t i = 0; i < m && uni; ++i) uni = (f_ptr[i + 1] - f_ptr[i] == npc);
      c->uniform_npc = uni ? (int)npc : 0;
    }
    // forward list continues with C's sym-upper entries (diagonal, then upper triangle of the CSR)
    for (int64_t j = 0; j < n; ++j)
      if (dC[j] != 0.0) { f_row.push_back((int)j); f_col.push_back((int)j); f_val.push_back(dC[j]); }
    for (int64_t j = 0; j < n; ++j)
      for (int e = c_rowptr[j]; e < c_rowptr[j + 1]; ++e)
        if (cents[e].col > j) { f_row.push_back((int)j); f_col.push_back(cents[e].col); f_val.push_back(cents[e].val); }
    c->nf_C = (int64_t)f_row.size() - c->nf_A;
    if (c->nf_C > 0) {
      const int64_t e1 = c->nf_A + c->nf_C;
      for (int64_t e = c->nf_A; e < e1; e += kChunk) { ch_beg.push_back(e); ch_end.push_back(std::min<int64_t>(e + kChunk, e1)); }
    }
    c->nchunk_all = (int64_t)ch_beg.size();
    std::vector<T> fv(f_val.size());
    for (size_t e = 0; e < f_val.size(); ++e) fv[e] = (T)f_val[e];
    ALORA_CUDA(c, upload(c, (void**)&c->f_ptr, f_ptr));
    ALORA_CUDA(c, upload(c, (void**)&c->f_row, f_row));
    ALORA_CUDA(c, upload(c, (void**)&c->f_col, f_col));
    ALORA_CUDA(c, upload(c, &c->f_val, fv));
    ALORA_CUDA(c, upload(c, (void**)&c->ch_beg, ch_beg));
    ALORA_CUDA(c, upload(c, (void**)&c->ch_end, ch_end));
    ALORA_CUDA(c, upload(c, (void**)&c->long_cons, long_cons));
    ALORA_CUDA(c, upload(c, (void**)&c->long_chptr, long_chptr));
    ALORA_CUDA(c, c->pool.alloc((void**)&c->ch_out, sizeof(double) * 3 * std::max<int64_t>(1, c->nchunk_A)));
    ALORA_CUDA(c, c->pool.alloc((void**)&c->part_long, sizeof(double) * kNStat * std::max(1, c->nlong_A)));
    ALORA_CUDA(c, c->pool.alloc((void**)&c->lam, sizeof(double) * std::max<int64_t>(1, m)));
  }
  // ---- low-rank cost term --------------------------------------------------------------------
  c->pC = P->pC;
  if (P->pC) {
    std::vector<T> U((size_t)n * P->pC);
    for (int p = 0; p < P->pC; ++p)
      for (int64_t j = 0; j < n; ++j) U[j * P->pC + p] = (T)P->C_U[(int64_t)p * n + j];
    ALORA_CUDA(c, upload(c, &c->U, U));
    c->s_host.assign(P->C_s, P->C_s + P->pC);
    ALORA_CUDA(c, upload(c, (void**)&c->s_dev, c->s_host));
    c->lr_grid = (int)std::min<int64_t>(2 * c->num_sms, std::max<int64_t>(1, n / 64));
    ALORA_CUDA(c, c->pool.alloc((void**)&c->lr_part, sizeof(double) * 2 * c->lr_grid * P->pC * c->lr_rmax));   // two matrices per launch
    ALORA_CUDA(c, c->pool.alloc((void**)&c->lr_ticket, sizeof(unsigned int) * 2));
    ALORA_CUDA(c, cudaMemset(c->lr_ticket, 0, sizeof(unsigned int) * 2));
    ALORA_CUDA(c, c->pool.alloc((void**)&c->TmR, sizeof(double) * P->pC * c->lr_rmax));
    ALORA_CUDA(c, c->pool.alloc((void**)&c->TmD, sizeof(double) * P->pC * c->lr_rmax));
    ALORA_CUDA(c, c->pool.alloc((void**)&c->Ts, sizeof(double) * P->pC * c->lr_rmax));
  }
  return ALORA_OK;
}

alora_status validate(const alora_problem* P, std::string& why) {
  if (!P) { why = "problem is NULL"; return ALORA_EINVAL; }
  if (P->n <= 0 || P->n >= INT32_MAX || P->m < 0 || P->m >= INT32_MAX || P->nnzC < 0 || P->nnzA < 0 || P->pC < 0 || P->pC > 8) {
    why = "bad sizes (need 0 < n < 2^31, 0 <= m < 2^31, 0 <= pC <= 8)"; return ALORA_EINVAL; }
  if ((P->nnzC && (!P->C_row || !P->C_col || !P->C_val)) || (P->nnzA && (!P->A_row || !P->A_col || !P->A_val)) ||
      !P->A_ptr || (P->m && !P->b) || (P->pC && (!P->C_U || !P->C_s))) { why = "NULL array"; return ALORA_EINVAL; }
  for (int64_t e = 0; e < P->nnzC; ++e)
    if (P->C_row[e] < 0 || P->C_row[e] > P->C_col[e] || P->C_col[e] >= P->n || !std::isfinite(P->C_val[e])) {
      why = "C entry " + std::to_string(e) + ": need 0 <= row <= col < n and a finite value"; return ALORA_EINVAL; }
  if (P->A_ptr[0] != 0 || P->A_ptr[P->m] != P->nnzA) { why = "A_ptr[0] != 0 or A_ptr[m] != nnzA"; return ALORA_EINVAL; }
  for (int64_t i = 0; i < P->m; ++i) {
    if (P->A_ptr[i + 1] < P->A_ptr[i]) { why = "A_ptr not monotone at " + std::to_string(i); return ALORA_EINVAL; }
    if (!std::isfinite(P->b[i])) { why = "b not finite at " + std::to_string(i); return ALORA_EINVAL; }
  }
  for (int64_t e = 0; e < P->nnzA; ++e)
    if (P->A_row[e] < 0 || P->A_row[e] > P->A_col[e] || P->A_col[e] >= P->n || !std::isfinite(P->A_val[e])) {
      why = "A entry " + std::to_string(e) + ": need 0 <= row <= col < n and a finite value"; return ALORA_EINVAL; }
  for (int64_t t = 0; t < (int64_t)P->pC * P->n; ++t)
    if (!std::isfinite(P->C_U[t])) { why = "C_U not finite"; return ALORA_EINVAL; }
  for (int p = 0; p < P->pC; ++p)
    if (!std::isfinite(P->C_s[p])) { why = "C_s not finite"; return ALORA_EINVAL; }
  return ALORA_OK;
}

thread_local std::string g_create_error;

}  // namespace
}  // namespace alora

using namespace alora;

extern "C" const char* alora_strerror(alora_status s) {
  switch (s) {
    case ALORA_OK: return "ok";
    case ALORA_EINVAL: return "invalid argument";
    case ALORA_ENOMEM: return "out of memory";
    case ALORA_ECUDA: return "CUDA error";
    case ALORA_ESTATE: return "call order violated";
    case ALORA_ENOTCONV: return "iteration cap reached";
  }
  return "unknown status";
}

extern "C" const char* alora_last_error(const alora_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

extern "C" void alora_destroy(alora_ctx* c) {
  if (!c) return;
  cudaSetDevice(c->device);
  free_solve_workspace(c);
  for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
  if (c->ev_eval) cudaEventDestroy(c->ev_eval);
  if (c->ev_down) cudaEventDestroy(c->ev_down);
  if (c->stream2) cudaStreamDestroy(c->stream2);
  c->pool.free_all();
  if (c->pinned) cudaFreeHost(c->pinned);
  if (c->pinR) cudaFreeHost(c->pinR);
  delete c;
}

extern "C" alora_status alora_create(const alora_problem* P, alora_dtype dtype, int device, void* cuda_stream,
                                     alora_ctx** out) {
  if (!out) return ALORA_EINVAL;
  *out = nullptr;
  std::string why;
  alora_status vs = validate(P, why);
  if (vs != ALORA_OK) { g_create_error = why; return vs; }
  if (dtype != ALORA_F32 && dtype != ALORA_F64) { g_create_error = "bad dtype"; return ALORA_EINVAL; }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
    g_create_error = "no such CUDA device (libalora has no CPU fallback)";
    cudaGetLastError();
    return ALORA_ECUDA;
  }
  if (cudaSetDevice(device) != cudaSuccess) { g_create_error = "cudaSetDevice failed"; return ALORA_ECUDA; }
  alora_ctx* c = new (std::nothrow) alora_ctx();
  if (!c) return ALORA_ENOMEM;
  c->device = device; c->stream = (cudaStream_t)cuda_stream; c->dtype = dtype;
  c->esz = dtype == ALORA_F32 ? 4 : 8; c->n = P->n; c->m = P->m;
  if (const char* e = std::getenv("ALORA_CW")) c->cw = std::atoi(e);   // measurement switch: 0 never, 1 default, 2 always
  if (const char* e = std::getenv("ALORA_SEL")) c->sel = std::atoi(e);       // measurement switch: dense line-search variant, 0 branches, 1 predicated loads, -1 by far share
  if (const char* e = std::getenv("ALORA_PDL")) c->pdl = std::atoi(e);       // measurement switch: programmatic dependent launch of the tiled kernel
  if (const char* e = std::getenv("ALORA_L2POL")) c->l2pol = std::atoi(e);   // measurement switch: L2 policies of the tiled kernel (RowArgs::l2pol), -1 = by size
  std::memset(c->occ_cache, 0, sizeof(c->occ_cache));
  std::memset(c->occ_ld, 0, sizeof(c->occ_ld));
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) == cudaSuccess) { c->num_sms = prop.multiProcessorCount; if (prop.l2CacheSize > 0) c->l2_bytes = (size_t)prop.l2CacheSize; }
  alora_status s;
  try {
    s = dtype == ALORA_F32 ? build<float>(c, P) : build<double>(c, P);
  } catch (const std::bad_alloc&) {
    s = fail(c, ALORA_ENOMEM, "host allocation failed while building the layouts");
  }
  auto bail = [&](alora_status st) { g_create_error = c->err; alora_destroy(c); return st; };
  if (s != ALORA_OK) return bail(s);
  c->part_cap = c->num_sms * 32;
  cudaError_t e = cudaSuccess;
  auto A = [&](void** p, size_t nb) { if (e == cudaSuccess) e = c->pool.alloc(p, nb); };
  A((void**)&c->part_rows, sizeof(double) * kNStat * c->part_cap);
  A((void**)&c->part_cons, sizeof(double) * kNStat * c->part_cap);
  A((void**)&c->part_chunk, sizeof(double) * kNStat * c->part_cap);
  A((void**)&c->stats_dev, sizeof(double) * kNStat * 4);
  A((void**)&c->z_int, sizeof(double) * std::max<int64_t>(1, c->m));
  A((void**)&c->lr_scal, sizeof(double) * 8);
  A((void**)&c->ticket, 16);
  if (e == cudaSuccess) e = cudaMemset(c->ticket, 0, 16);
  if (e == cudaSuccess) e = cudaHostAlloc((void**)&c->pinned, sizeof(double) * (64 + 2 * 8 * 256), cudaHostAllocDefault);
  if (e != cudaSuccess) {
    fail(c, ALORA_ECUDA, cudaGetErrorString(e));
    return bail(e == cudaErrorMemoryAllocation ? ALORA_ENOMEM : ALORA_ECUDA);
  }
  c->ls_dev = c->stats_dev + kNStat;
  c->mv_dev = c->stats_dev + 2 * kNStat;
  // the uploads and memsets above ran on the legacy default stream; the ctx stream may be a non-blocking one that
  // is not ordered against it, so everything is made complete before the first call can enqueue work
  if (cudaDeviceSynchronize() != cudaSuccess) { fail(c, ALORA_ECUDA, "cudaDeviceSynchronize failed at the end of alora_create"); return bail(ALORA_ECUDA); }
  *out = c;
  return ALORA_OK;
}

extern "C" alora_status alora_info(const alora_ctx* c, int64_t info[16]) {
  if (!c || !info) return ALORA_EINVAL;
  for (int i = 0; i < 16; ++i) info[i] = 0;
  info[0] = c->cls; info[1] = c->n; info[2] = c->m; info[3] = c->c_nnz; info[4] = c->a_nnz; info[5] = c->nf_A;
  info[6] = c->nlong_A; info[7] = c->launches; info[8] = (int64_t)c->pool.bytes; info[9] = c->num_sms;
  info[10] = c->nf_C;
  return ALORA_OK;
}

extern "C" alora_status alora_set_dual(alora_ctx* c, const double* y_dev, double sigma) {
  if (!c) return ALORA_EINVAL;
  if ((!y_dev && c->m > 0) || !(sigma > 0.0) || !std::isfinite(sigma))
    return fail(c, ALORA_EINVAL, "alora_set_dual: need y_dev != NULL and finite sigma > 0");
  c->y = y_dev; c->sigma = sigma; c->have_dual = true; c->have_eval = false; c->last_eval_R = nullptr;
  return ALORA_OK;
}
