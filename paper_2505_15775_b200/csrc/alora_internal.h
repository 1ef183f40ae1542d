// alora_internal.h -- the context behind include/alora.h (host side).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/alora.h"
#include "dispatch.h"

namespace alora {

// device array with byte accounting
struct DevPool {
  std::vector<void*> ptrs;
  std::vector<size_t> sizes;
  size_t bytes = 0;
  cudaError_t alloc(void** p, size_t nbytes) {
    *p = nullptr;
    if (nbytes == 0) nbytes = 16;
    cudaError_t e = cudaMalloc(p, nbytes);
    if (e == cudaSuccess) { ptrs.push_back(*p); sizes.push_back(nbytes); bytes += nbytes; }
    return e;
  }
  void release(void* p) {
    if (!p) return;
    for (size_t i = 0; i < ptrs.size(); ++i)
      if (ptrs[i] == p) { cudaFree(p); bytes -= sizes[i]; ptrs[i] = nullptr; sizes[i] = 0; }
  }
  void free_all() {
    for (void* p : ptrs) if (p) cudaFree(p);
    ptrs.clear(); sizes.clear(); bytes = 0;
  }
};

struct SolveWorkspace;  // alora_solve.cu

}  // namespace alora

struct alora_ctx {
  int device = 0;
  cudaStream_t stream = nullptr;
  alora_dtype dtype = ALORA_F32;
  size_t esz = 4;
  int64_t n = 0, m = 0;
  int cls = 0;  // 0: diagonal class (one fused pass), 1: general (forward + adjoint)
  int num_sms = 148;
  std::string err;
  alora::DevPool pool;

  // C: diagonal + off-diagonal full-pattern CSR (columns ascending within a row)
  int* c_rowptr = nullptr; int* c_col = nullptr; void* c_val = nullptr; void* dC = nullptr;
  int64_t c_nnz = 0;
  // diagonal class: constraint of row j (-1: none) and its coefficient; null = identity / ones
  int* dcons = nullptr; void* da = nullptr;
  // identity diagonal class: padded ELL blocks (rows_tiled.cuh): kUN first neighbours per row, kUNL last
  // upper-triangle neighbours per row, and per 32-row block a flag "some row has more"
  int cw = 1;              // general class, cooperative entry / row kernels (k_ent_cw, k_rows_cw): 1 = where they pay (use_cw), 0 = never, 2 = always (ALORA_CW)
  int occ_cw[3][6] = {};
  int64_t ell_hist[2][34] = {};   // used ELL slots (0: f + grad / adjoint block, 1: line-search block) by bit length of |col - row|
  size_t l2_bytes = 126u << 20;
  int sel = -1;            // dense variants of the tiled kernel: predicated neighbour loads (1), branches (0), -1 = by the share of far neighbours (ALORA_SEL)
  int pdl = 1;             // hot-path kernels launched with programmatic stream serialisation: 0 never, 1 by use_pdl() (alora_ctx.cu), 2 always (ALORA_PDL)
  int l2pol = -1;          // L2 cache policies of the tiled row kernel (RowArgs::l2pol); -1: chosen per call from the sizes (ALORA_L2POL)
  bool ell_wide = false;   // 8 / 6 slots per row instead of 4 / 3 (more than 10 % of the rows have degree > 4)
  int* ell_col = nullptr; void* ell_val = nullptr;
  int* ellu_col = nullptr; void* ellu_val = nullptr;
  // general class: row-oriented full pattern of the constraints
  int* a_rowptr = nullptr; int* a_col = nullptr; void* a_val = nullptr; int* a_cons = nullptr;
  int64_t a_nnz = 0;
  // heavy C rows (> kHeavyRow entries) cut into segments for k_rows_seg / k_rows_ep
  int nseg = 0, nheavy = 0; int* seg_row = nullptr; int* seg_beg = nullptr; int* seg_end = nullptr;
  int* heavy_rows = nullptr; int* heavy_segptr = nullptr; void* seg_out = nullptr; double* seg_cx = nullptr;
  size_t seg_out_bytes = 0;   // seg_out is sized on first use for the row length in use (nseg * pitch elements)
  int uniform_npc = 0;         // > 1: every constraint has exactly this many stored entries and it divides 32
  bool single_entry = false;   // every constraint has exactly one stored entry: thread-per-constraint forward (k_cons1)
  bool short_cons = false;     // at most 8 stored entries per constraint on average: thread-per-constraint forward too
  bool ep = false;       // general class, >= 8 entries per row on average: warp-per-row adjoint for single vectors
  int* row_perm = nullptr;  // general class, skewed row lengths: rows by decreasing work (k_rows walks this order)
  bool ep_wide = false;  // >= 96 entries per row on average (matrix completion): warp-per-row adjoint for every r
  // forward list: coalesced constraint entries [0, nf_A), then C's sym-upper entries [nf_A, nf_A+nf_C)
  int64_t* f_ptr = nullptr; int* f_row = nullptr; int* f_col = nullptr; void* f_val = nullptr;
  int64_t nf_A = 0, nf_C = 0;
  // chunks of long constraints (first nchunk_A) and of C (the rest); slots: long constraints, then C
  int64_t* ch_beg = nullptr; int64_t* ch_end = nullptr; int64_t nchunk_A = 0, nchunk_all = 0;
  int* long_cons = nullptr; int64_t* long_chptr = nullptr; int nlong_A = 0;
  double* ch_out = nullptr;
  void* e_out = nullptr;      // per-entry sums of the cooperative forward evaluator (nf_A x 3, ctx dtype), on first use
  // vectors
  double* b = nullptr; const double* y = nullptr; double sigma = 0.0; bool have_dual = false;
  double* z_int = nullptr; double* lam = nullptr; const double* z_last = nullptr;
  double normb = 0.0, normC = 0.0;
  // low-rank cost
  int pC = 0; void* U = nullptr; double* s_dev = nullptr; std::vector<double> s_host;
  double* lr_part = nullptr; double* TmR = nullptr; double* TmD = nullptr; double* Ts = nullptr; double* lr_scal = nullptr;
  int lr_grid = 0; int lr_rmax = 256; unsigned int* lr_ticket = nullptr;   // k_lowrank: one ticket word per matrix of a launch
  // partial sums / results
  int part_cap = 0;
  double* part_rows = nullptr; double* part_cons = nullptr; double* part_long = nullptr; double* part_chunk = nullptr;
  double* stats_dev = nullptr; double* ls_dev = nullptr; double* mv_dev = nullptr;
  unsigned int* ticket = nullptr;   // FinArgs::ticket (kernels.cuh), zero between launches
  double* pinned = nullptr;  // 64 doubles
  bool have_eval = false, have_ls = false;
  int last_eval_r = 0, last_ls_r = 0;
  const void* last_eval_R = nullptr; int64_t last_eval_ld = 0;   // what a warm alora_linesearch must match
  const void* last_eval_G = nullptr;                              // gradient that evaluation wrote (null: value-only call)
  bool ls_used_g = false;                                         // the last line search took p1 = <G,D> from that gradient
  bool ls_warm = false; double* ls_warm_stats = nullptr;          // copy of the evaluation's scalars taken by a warm call
  double* lam_auto = nullptr;   // diagonal class: lambda of the last evaluation, formed on demand (mu_dev == NULL)
  int64_t launches = 0;
  // staging for alora_eval_host
  void* stageR = nullptr; void* stageG = nullptr; size_t stage_bytes = 0;
  void* stageD = nullptr; void* stageV = nullptr; void* stageW = nullptr; size_t stage2_bytes = 0;   // alora_step_host
  cudaStream_t stream2 = nullptr; cudaEvent_t ev_eval = nullptr, ev_down = nullptr;                  // second copy stream
  void* pinR = nullptr; size_t pin_bytes = 0;
  // occupancy cache [vec idx][shape][kind]
  int occ_cache[3][7][12];
  int64_t occ_ld[3][7][4];   // ld for which the tiled-kernel occupancy was computed
  alora::SolveWorkspace* ws = nullptr;
  // optional CUDA-event timing of the dominant kernel of alora_eval (bench.py roofline)
  bool timing = false; int timing_every = 1; int64_t timing_calls = 0; std::vector<cudaEvent_t> ev; size_t ev_used = 0;
};

namespace alora {

alora_status fail(alora_ctx* c, alora_status s, const std::string& msg);
#define ALORA_CUDA(c, expr)                                                                        \
  do {                                                                                             \
    cudaError_t e__ = (expr);                                                                      \
    if (e__ != cudaSuccess)                                                                        \
      return alora::fail((c), e__ == cudaErrorMemoryAllocation ? ALORA_ENOMEM : ALORA_ECUDA,      \
                         std::string(#expr) + ": " + cudaGetErrorString(e__));                     \
  } while (0)

// alora_ctx.cu
alora_status stats_enqueue(alora_ctx* c, int r_lowrank);                    // scalars of the last evaluation: enqueue the copies ...
void stats_finish(alora_ctx* c, int r_lowrank, double stats[8]);          // ... and assemble them after a synchronise
alora_status resolve_mu(alora_ctx* c, const double** mu, const char* who);   // NULL -> lambda of the last alora_eval
int pick_vec(const alora_ctx* c, int64_t ld, const void* p0, const void* p1, const void* p2);
void free_solve_workspace(alora_ctx* c);

}  // namespace alora
