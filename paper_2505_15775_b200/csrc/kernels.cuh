// kernels.cuh -- templated sm_100a kernels of the ALM-BM hot path.
//
// Two kernel families, both HBM-bound gather/stream kernels (no dense contraction => no tensor cores):
//   k_rows : one sub-warp group of GS lanes per row j of R (thin row, r = 10..40 elements, held in
//            registers as NIT vectors of VEC elements per lane).  Streams the row-oriented CSR,
//            gathers neighbour rows with vector loads, writes the output row, and accumulates every
//            scalar of the evaluation lane-locally in fp64 (one block reduction at the very end).
//              ROWS_FUSED_EVAL : "diagonal" class (MaxCut): z_j = a_j |R_j|^2 is row-local, so
//                                z, q, lambda, G = 2 S(lambda) R, <C,RR^T>, y.q, |q|^2, |G|^2, <G,R>
//                                come out of ONE pass                       (a1-a4 fused)
//              ROWS_ADJ        : weighted-adjoint SpMM  Out = scale * (C - sum_i w_i A_i) X with the
//                                weights w gathered by constraint id        (a3; a6 with scale = 1)
//              ROWS_LS_FUSED   : line-search sums for the diagonal class    (a5)
//   k_cons : SDDMM-style forward evaluator, one group per constraint (or per chunk of a long
//            constraint): sum_e w_e a_e <R_j,R_k>  and the bilinear forms with D   (a1, a2, a5)
// Sums across rows / constraints are fp64 and two-stage (per-block partials, then one ordered
// reduction), so results do not depend on block scheduling.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace alora {

// Programmatic dependent launch.  Every kernel of the hot path starts with ALORA_GRID_DEP(): it waits until the kernels
// before it in the stream have completed and flushed (it reads what they wrote), and lets its own successor become
// resident.  Both instructions are no-ops in a plain launch.  launch_k launches with programmatic stream serialisation
// when `pdl` is set (alora_ctx::pdl), so that the blocks of the next kernel are scheduled while this one drains.
#define ALORA_GRID_DEP()                                            \
  do {                                                              \
    asm volatile("griddepcontrol.wait;" ::: "memory");              \
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); \
  } while (0)
template <typename... KA, typename... A>
inline cudaError_t launch_k(bool pdl, void (*k)(KA...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, A&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, k, static_cast<KA>(args)...);
}

constexpr int kBlock = 256;
constexpr int kGeneralRow = 512;      // a C row with more entries sends a diagonal-class problem down the general path
constexpr int kHeavyRow = 128;        // general path: C rows with more entries are cut into segments of this many entries
constexpr int kLongThreshold = 64;   // constraints with more stored entries are split into chunks
constexpr int kChunk = 16;           // entries per chunk of a long constraint / of C's sym-upper list
// diagonal class: ELL slots per row (first neighbours; for the line search: last upper-triangle neighbours), see
// rows_tiled.cuh.  Two widths, chosen per problem in alora_create: narrow for degree <= 4 graphs (grids, ring +
// matchings), wide for mesh-like graphs of degree 6..8.
__host__ __device__ constexpr int ell_slots(bool wide) { return wide ? 8 : 4; }
__host__ __device__ constexpr int ell_slots_ls(bool wide) { return wide ? 6 : 3; }

enum RowsMode { ROWS_FUSED_EVAL = 0, ROWS_ADJ = 1, ROWS_LS_FUSED = 2, ROWS_LS_WARM = 3 };   // LS_WARM: k_rows_tiled only (RowArgs::X3)
enum ConsMode { CONS_EVAL = 0, CONS_LS = 1 };

// stat slots written by the kernels (per-block partial rows have this many doubles)
constexpr int kNStat = 16;
enum EvalStat { ES_CX = 0, ES_YQ = 1, ES_QQ = 2, ES_GG = 3, ES_GR = 4, ES_LZ = 5 };
enum LsStat { LS_CRR = 0, LS_CRD = 1, LS_CDD = 2, LS_YQ = 3, LS_YQ1 = 4, LS_YQ2 = 5, LS_QQ = 6,
              LS_QQ1 = 7, LS_QQ2 = 8, LS_Q11 = 9, LS_Q12 = 10, LS_Q22 = 11 };

// Fused final reduction: the LAST kernel of a call also sums the per-block partial rows of the call (its own
// and those written by the kernels launched before it on the stream) into out[0..16).  Every block publishes
// its row, takes a ticket, and the block that draws the last ticket does the sum in a fixed order, so the result
// does not depend on which block that is.  out == nullptr: the kernel only writes its partial rows.
struct FinArgs {
  const double* p[3]; int n[3];   // up to three regions of partial rows ([n][kNStat])
  double* out;                    // [kNStat]
  unsigned int* ticket;           // zero before the launch; reset by the finishing block
};

template <typename T> struct RowArgs {
  int64_t n; int r; int64_t ld; int nvec; int exact;  // exact: r == nvec*VEC (no tail masking)
  const T* X;    // R (or V)
  const T* X2;   // D (ROWS_LS_FUSED)
  const T* X3;   // k_rows_tiled<ROWS_LS_WARM>: G = grad f(R) of the evaluation on record
  T* Out;        // G / W, may be null
  const int* c_rowptr; const int* c_col; const T* c_val; const T* dC;  // off-diagonal C (full pattern) + diag
  const int* dcons; const T* da;       // diagonal class: constraint on row j and its coefficient (null: j / 1)
  const int* a_rowptr; const int* a_col; const T* a_val; const int* a_cons;  // general class, full pattern
  const double* y; const double* b; double sigma;
  const double* w;   // ROWS_ADJ weights (lambda or mu), fp64[m]
  double* z;         // ROWS_FUSED_EVAL: z out (fp64[m]) or null
  int pC; const T* U; const double* Ts;  // low-rank cost: U n x pC row-major, Ts[p][r] = s_p (U^T X)_p
  double scale;
  int diag_class;    // ROWS_ADJ: 1 = constraints are the per-row diagonal ones, 0 = use a_* CSR
  double* partials;  // [gridDim.x][kNStat]
  FinArgs fin;
  int64_t row_begin; // k_rows: first row handled (rows [row_begin, n))
  int64_t tiles;     // k_rows_tiled: number of full row tiles handled (rows [0, tiles * TR))
  // k_rows_tiled: padded ELL block of the mode (kUN first neighbours, or kUNL last upper-triangle neighbours
  // for the line search): slot u of row j at [j * NU + u]; sign bit of the first slot's column: the row has more
  // neighbours than slots (walk the CSR tail)
  const int* ell_col; const T* ell_val;
  // k_rows_ep: C rows with more than kHeavyRow entries are cut into segments of <= kHeavyRow entries that
  // k_rows_seg sums first (seg_out[s][nvec * VEC], seg_cx[s]); heavy_rows (ascending) / heavy_segptr list them per row
  int nseg, nheavy; const int* seg_row; const int* seg_beg; const int* seg_end;
  const int* heavy_rows; const int* heavy_segptr; T* seg_out; double* seg_cx;
  // optional processing order of the rows (general class, skewed degrees): position -> row, heaviest rows first
  const int* perm;
  // k_rows_tiled: L2 cache policies (bit 0: per-row metadata copies evict_first; bit 1: X / X2 tile copies evict_first;
  // bit 2: gathered neighbour rows evict_last; bit 3: output rows evict_first; bit 5: X tile copies evict_last)
  int l2pol;
  int pdl;   // host only: programmatic dependent launch (alora_ctx::pdl)
};

template <typename T> struct ConsArgs {
  int64_t n; int r; int64_t ld; int nvec; int exact;
  const T* X; const T* X2;
  int64_t m;                      // number of real constraints
  const int64_t* ptr;             // m+1 (short kernel)
  const int* e_row; const int* e_col; const T* e_val;  // forward entries (constraints, then C)
  const double* y; const double* b; double sigma;
  double* z; double* lam;         // CONS_EVAL outputs
  // chunk kernel
  int64_t nchunk; const int64_t* ch_beg; const int64_t* ch_end;
  int64_t nchunk_A;               // chunks [0, nchunk_A) belong to long constraints, the rest to C's sym-upper list
  double* ch_out;                 // [nchunk_A][3]
  double* part_chunk;             // chunk kernel: per-block partial rows (sums over C's chunks)
  double* partials;
  FinArgs fin;
  // cooperative forward evaluator (k_ent_cw / k_cons_fin / k_long_fin_e): entries [0, nent) are walked, the first nf_A
  // of them belong to constraints (their per-entry sums go to e_out[e][K], K = 1 or 3), the rest to C's sym-upper list
  int64_t nent, nf_A; T* e_out;
  int npc;                        // > 1: every constraint has exactly npc entries (npc divides 32): k_ent_cw finishes them itself
  const int* long_cons;           // ids of the constraints with more than kLongThreshold entries (one block each)
  int pdl;                        // host only: programmatic dependent launch (alora_ctx::pdl)
};

// ---------------------------------------------------------------------------------------------
template <typename T, int VEC> struct alignas(sizeof(T) * VEC) Pack { T v[VEC]; };

// Read-only row loads.  ALORA_LD_L2HINT (default on): ld.global.nc with the L2::64B prefetch-size hint -- measured on
// config 4 (random 40-byte row gathers from a 671 MB R): 1 150 -> 1 109 us for the f + grad kernel; plain
// ld.global.nc (__ldg), .L1::no_allocate, .cg and .cs were equal or slower (profiles/r1t_README.md).
#ifndef ALORA_LD_L2HINT
#define ALORA_LD_L2HINT 1
#endif
#if ALORA_LD_L2HINT
#define ALORA_LD_NC "ld.global.nc.L2::64B"
#else
#define ALORA_LD_NC "ld.global.nc"
#endif
template <typename T, int VEC> __device__ __forceinline__ Pack<T, VEC> ldg_pack(const T* p);
template <> __device__ __forceinline__ Pack<float, 4> ldg_pack<float, 4>(const float* p) {
  Pack<float, 4> o;
  asm(ALORA_LD_NC ".v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(o.v[0]), "=f"(o.v[1]), "=f"(o.v[2]), "=f"(o.v[3]) : "l"(p));
  return o; }
template <> __device__ __forceinline__ Pack<float, 2> ldg_pack<float, 2>(const float* p) {
  Pack<float, 2> o;
  asm(ALORA_LD_NC ".v2.f32 {%0,%1}, [%2];" : "=f"(o.v[0]), "=f"(o.v[1]) : "l"(p));
  return o; }
template <> __device__ __forceinline__ Pack<float, 1> ldg_pack<float, 1>(const float* p) {
  Pack<float, 1> o;
  asm(ALORA_LD_NC ".f32 %0, [%1];" : "=f"(o.v[0]) : "l"(p));
  return o; }
template <> __device__ __forceinline__ Pack<double, 2> ldg_pack<double, 2>(const double* p) {
  Pack<double, 2> o;
  asm(ALORA_LD_NC ".v2.f64 {%0,%1}, [%2];" : "=d"(o.v[0]), "=d"(o.v[1]) : "l"(p));
  return o; }
template <> __device__ __forceinline__ Pack<double, 1> ldg_pack<double, 1>(const double* p) {
  Pack<double, 1> o;
  asm(ALORA_LD_NC ".f64 %0, [%1];" : "=d"(o.v[0]) : "l"(p));
  return o; }

template <typename T, int VEC> __device__ __forceinline__ void st_pack(T* p, const Pack<T, VEC>& x) {
  *reinterpret_cast<Pack<T, VEC>*>(p) = x;
}

// L2 cache policies (createpolicy) for the loads / stores / bulk copies of the tiled row kernel: kind 0 = evict_normal
// (the default behaviour), 1 = evict_first (data read or written once per launch: slots, y, b, outputs), 2 = evict_last
// (data other rows will gather again: the rows of X).  The policy is an operand, so one kernel serves all settings.
__device__ __forceinline__ uint64_t l2_policy(int kind) {
  uint64_t p;
  if (kind == 1) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  else if (kind == 2) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
  else asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
  return p;
}
#if ALORA_LD_L2HINT
#define ALORA_LD_NCP "ld.global.nc.L2::cache_hint.L2::64B"
#else
#define ALORA_LD_NCP "ld.global.nc.L2::cache_hint"
#endif
template <typename T, int VEC> __device__ __forceinline__ Pack<T, VEC> ldg_pack_pol(const T* p, uint64_t pol);
template <> __device__ __forceinline__ Pack<float, 4> ldg_pack_pol<float, 4>(const float* p, uint64_t pol) {
  Pack<float, 4> o;
  asm(ALORA_LD_NCP ".v4.f32 {%0,%1,%2,%3}, [%4], %5;" : "=f"(o.v[0]), "=f"(o.v[1]), "=f"(o.v[2]), "=f"(o.v[3]) : "l"(p), "l"(pol));
  return o; }
template <> __device__ __forceinline__ Pack<float, 2> ldg_pack_pol<float, 2>(const float* p, uint64_t pol) {
  Pack<float, 2> o;
  asm(ALORA_LD_NCP ".v2.f32 {%0,%1}, [%2], %3;" : "=f"(o.v[0]), "=f"(o.v[1]) : "l"(p), "l"(pol));
  return o; }
template <> __device__ __forceinline__ Pack<float, 1> ldg_pack_pol<float, 1>(const float* p, uint64_t pol) {
  Pack<float, 1> o;
  asm(ALORA_LD_NCP ".f32 %0, [%1], %2;" : "=f"(o.v[0]) : "l"(p), "l"(pol));
  return o; }
template <> __device__ __forceinline__ Pack<double, 2> ldg_pack_pol<double, 2>(const double* p, uint64_t pol) {
  Pack<double, 2> o;
  asm(ALORA_LD_NCP ".v2.f64 {%0,%1}, [%2], %3;" : "=d"(o.v[0]), "=d"(o.v[1]) : "l"(p), "l"(pol));
  return o; }
template <> __device__ __forceinline__ Pack<double, 1> ldg_pack_pol<double, 1>(const double* p, uint64_t pol) {
  Pack<double, 1> o;
  asm(ALORA_LD_NCP ".f64 %0, [%1], %2;" : "=d"(o.v[0]) : "l"(p), "l"(pol));
  return o; }
// One pack from shared memory (ps != 0: 32-bit shared address sa) or from global memory (pg != 0: read-only path with
// the L2::64B fetch size and cache policy pol), or zeros (neither) -- as two PREDICATED loads instead of a branch: a
// warp whose lanes disagree (one row's neighbour sits in the staged tile, the next row's does not) otherwise pays a
// BSSY / BRA / BSYNC group per neighbour load.  volatile: the shared-memory stage is rewritten between iterations.
template <typename T, int VEC> __device__ __forceinline__ Pack<T, VEC> ld_sel(uint32_t sa, const T* gp, int ps, int pg, uint64_t pol);
template <> __device__ __forceinline__ Pack<float, 4> ld_sel<float, 4>(uint32_t sa, const float* gp, int ps, int pg, uint64_t pol) {
  Pack<float, 4> o;
  asm volatile("{\n .reg .pred ps, pg;\n setp.ne.s32 ps, %6, 0;\n setp.ne.s32 pg, %7, 0;\n mov.f32 %0, 0f00000000;\n mov.f32 %1, 0f00000000;\n mov.f32 %2, 0f00000000;\n mov.f32 %3, 0f00000000;\n @ps ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];\n @pg " ALORA_LD_NCP ".v4.f32 {%0,%1,%2,%3}, [%5], %8;\n}"
               : "=&f"(o.v[0]), "=&f"(o.v[1]), "=&f"(o.v[2]), "=&f"(o.v[3]) : "r"(sa), "l"(gp), "r"(ps), "r"(pg), "l"(pol));
  return o; }
template <> __device__ __forceinline__ Pack<float, 2> ld_sel<float, 2>(uint32_t sa, const float* gp, int ps, int pg, uint64_t pol) {
  Pack<float, 2> o;
  asm volatile("{\n .reg .pred ps, pg;\n setp.ne.s32 ps, %4, 0;\n setp.ne.s32 pg, %5, 0;\n mov.f32 %0, 0f00000000;\n mov.f32 %1, 0f00000000;\n @ps ld.shared.v2.f32 {%0,%1}, [%2];\n @pg " ALORA_LD_NCP ".v2.f32 {%0,%1}, [%3], %6;\n}"
               : "=&f"(o.v[0]), "=&f"(o.v[1]) : "r"(sa), "l"(gp), "r"(ps), "r"(pg), "l"(pol));
  return o; }
template <> __device__ __forceinline__ Pack<float, 1> ld_sel<float, 1>(uint32_t sa, const float* gp, int ps, int pg, uint64_t pol) {
  Pack<float, 1> o;
  asm volatile("{\n .reg .pred ps, pg;\n setp.ne.s32 ps, %3, 0;\n setp.ne.s32 pg, %4, 0;\n mov.f32 %0, 0f00000000;\n @ps ld.shared.f32 %0, [%1];\n @pg " ALORA_LD_NCP ".f32 %0, [%2], %5;\n}"
               : "=&f"(o.v[0]) : "r"(sa), "l"(gp), "r"(ps), "r"(pg), "l"(pol));
  return o; }
template <> __device__ __forceinline__ Pack<double, 2> ld_sel<double, 2>(uint32_t sa, const double* gp, int ps, int pg, uint64_t pol) {
  Pack<double, 2> o;
  asm volatile("{\n .reg .pred ps, pg;\n setp.ne.s32 ps, %4, 0;\n setp.ne.s32 pg, %5, 0;\n mov.f64 %0, 0d0000000000000000;\n mov.f64 %1, 0d0000000000000000;\n @ps ld.shared.v2.f64 {%0,%1}, [%2];\n @pg " ALORA_LD_NCP ".v2.f64 {%0,%1}, [%3], %6;\n}"
               : "=&d"(o.v[0]), "=&d"(o.v[1]) : "r"(sa), "l"(gp), "r"(ps), "r"(pg), "l"(pol));
  return o; }
template <> __device__ __forceinline__ Pack<double, 1> ld_sel<double, 1>(uint32_t sa, const double* gp, int ps, int pg, uint64_t pol) {
  Pack<double, 1> o;
  asm volatile("{\n .reg .pred ps, pg;\n setp.ne.s32 ps, %3, 0;\n setp.ne.s32 pg, %4, 0;\n mov.f64 %0, 0d0000000000000000;\n @ps ld.shared.f64 %0, [%1];\n @pg " ALORA_LD_NCP ".f64 %0, [%2], %5;\n}"
               : "=&d"(o.v[0]) : "r"(sa), "l"(gp), "r"(ps), "r"(pg), "l"(pol));
  return o; }
template <typename T, int VEC> __device__ __forceinline__ void st_pack_pol(T* p, const Pack<T, VEC>& x, uint64_t pol);
template <> __device__ __forceinline__ void st_pack_pol<float, 4>(float* p, const Pack<float, 4>& x, uint64_t pol) {
  asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1,%2,%3,%4}, %5;" ::"l"(p), "f"(x.v[0]), "f"(x.v[1]), "f"(x.v[2]), "f"(x.v[3]), "l"(pol) : "memory"); }
template <> __device__ __forceinline__ void st_pack_pol<float, 2>(float* p, const Pack<float, 2>& x, uint64_t pol) {
  asm volatile("st.global.L2::cache_hint.v2.f32 [%0], {%1,%2}, %3;" ::"l"(p), "f"(x.v[0]), "f"(x.v[1]), "l"(pol) : "memory"); }
template <> __device__ __forceinline__ void st_pack_pol<float, 1>(float* p, const Pack<float, 1>& x, uint64_t pol) {
  asm volatile("st.global.L2::cache_hint.f32 [%0], %1, %2;" ::"l"(p), "f"(x.v[0]), "l"(pol) : "memory"); }
template <> __device__ __forceinline__ void st_pack_pol<double, 2>(double* p, const Pack<double, 2>& x, uint64_t pol) {
  asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1,%2}, %3;" ::"l"(p), "d"(x.v[0]), "d"(x.v[1]), "l"(pol) : "memory"); }
template <> __device__ __forceinline__ void st_pack_pol<double, 1>(double* p, const Pack<double, 1>& x, uint64_t pol) {
  asm volatile("st.global.L2::cache_hint.f64 [%0], %1, %2;" ::"l"(p), "d"(x.v[0]), "l"(pol) : "memory"); }

template <int GS> __device__ __forceinline__ unsigned group_mask() {
  if (GS >= 32) return 0xffffffffu;
  return ((1u << GS) - 1u) << (((threadIdx.x & 31) / GS) * GS);
}
template <int GS> __device__ __forceinline__ double group_sum(double v, unsigned mask) {
#pragma unroll
  for (int o = GS / 2; o > 0; o >>= 1) v += __shfl_xor_sync(mask, v, o);
  return v;
}
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Ordered block reduction of NST per-thread fp64 partials -> out[0..NST)
template <int NST> __device__ __forceinline__ void block_reduce_store(double (&st)[NST], double* out) {
  __shared__ double sm[NST][kBlock / 32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int s = 0; s < NST; ++s) {
    double v = warp_sum(st[s]);
    if (lane == 0) sm[s][warp] = v;
  }
  __syncthreads();
  if (threadIdx.x < kNStat) {  // unused slots of the partial row are written as zero
    double v = 0.0;
    if (threadIdx.x < NST) {
#pragma unroll
      for (int wv = 0; wv < kBlock / 32; ++wv) v += sm[threadIdx.x][wv];
    }
    out[threadIdx.x] = v;
  }
}

// See FinArgs.  Called by every thread of the block after the block's partial row has been written (needs
// blockDim.x >= 256).  Thread t < 256 owns stat t % 16 and the rows t / 16, t / 16 + 16, ... of each region; the 16
// row slots are then summed in order through shared memory.
#ifndef ALORA_FIN_LOADS
#define ALORA_FIN_LOADS 16
#endif
constexpr int kFinLoads = ALORA_FIN_LOADS;   // 444 partial rows / 16 row slots = 28 loads per thread: two round trips instead of four
__device__ __forceinline__ void finish_partials(const FinArgs& f) {
  if (!f.out) return;
  __shared__ unsigned int s_last;
  __shared__ double s_fin[256];
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) s_last = (atomicAdd(f.ticket, 1u) == gridDim.x - 1) ? 1u : 0u;
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  if (threadIdx.x < 256) {
    const int s = threadIdx.x & (kNStat - 1), slot = threadIdx.x / kNStat;
    constexpr int NSLOT = 256 / kNStat;
    double v = 0.0;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const double* p = f.p[k];
      const int n = f.n[k];
      for (int i = slot; i < n; i += kFinLoads * NSLOT) {   // kFinLoads independent (predicated) loads in flight per round trip
        double t[kFinLoads];
#pragma unroll
        for (int u = 0; u < kFinLoads; ++u) t[u] = (i + u * NSLOT < n) ? __ldcg(p + (int64_t)(i + u * NSLOT) * kNStat + s) : 0.0;
#pragma unroll
        for (int u = 0; u < kFinLoads; ++u) v += t[u];
      }
    }
    s_fin[threadIdx.x] = v;
  }
  __syncthreads();
  if (threadIdx.x < kNStat) {
    double t = 0.0;
    for (int k = 0; k < 256 / kNStat; ++k) t += s_fin[k * kNStat + threadIdx.x];
    f.out[threadIdx.x] = t;
  }
  if (threadIdx.x == 0) *f.ticket = 0u;
}

// Row vector held by one lane: NIT packs of VEC elements, pack index vi = lane + it*GS.
template <typename T, int VEC, int GS, int NIT> struct RowReg {
  Pack<T, VEC> p[NIT];
  __device__ __forceinline__ void zero() {
#pragma unroll
    for (int it = 0; it < NIT; ++it)
#pragma unroll
      for (int i = 0; i < VEC; ++i) p[it].v[i] = T(0);
  }
  // load row `base` (pointer to the first element of the row); masks the tail beyond r
  __device__ __forceinline__ void load(const T* base, int lane, int nvec, int r, int exact) {
#pragma unroll
    for (int it = 0; it < NIT; ++it) {
      const int vi = lane + it * GS;
      if (vi < nvec) {
        p[it] = ldg_pack<T, VEC>(base + vi * VEC);
        if (VEC > 1 && !exact && vi == nvec - 1) {
#pragma unroll
          for (int i = 0; i < VEC; ++i) if (vi * VEC + i >= r) p[it].v[i] = T(0);
        }
      } else {
#pragma unroll
        for (int i = 0; i < VEC; ++i) p[it].v[i] = T(0);
      }
    }
  }
  __device__ __forceinline__ void store(T* base, int lane, int nvec, int r, int exact) const {
#pragma unroll
    for (int it = 0; it < NIT; ++it) {
      const int vi = lane + it * GS;
      if (vi < nvec) {
        if (VEC > 1 && !exact && vi == nvec - 1) {
#pragma unroll
          for (int i = 0; i < VEC; ++i) if (vi * VEC + i < r) base[vi * VEC + i] = p[it].v[i];
        } else {
          st_pack<T, VEC>(base + vi * VEC, p[it]);
        }
      }
    }
  }
  __device__ __forceinline__ void axpy(T a, const RowReg& x) {
#pragma unroll
    for (int it = 0; it < NIT; ++it)
#pragma unroll
      for (int i = 0; i < VEC; ++i) p[it].v[i] = fma(a, x.p[it].v[i], p[it].v[i]);
  }
  __device__ __forceinline__ T dot(const RowReg& x) const {  // lane-local part of the dot product
    T s = T(0);
#pragma unroll
    for (int it = 0; it < NIT; ++it)
#pragma unroll
      for (int i = 0; i < VEC; ++i) s = fma(p[it].v[i], x.p[it].v[i], s);
    return s;
  }
};

// acc += sum_e val[e] * X[col[e], :]   (unrolled so several gathers are in flight per group)
template <typename T, int VEC, int GS, int NIT>
__device__ __forceinline__ void gather_axpy(RowReg<T, VEC, GS, NIT>& acc, const T* __restrict__ X, int64_t ld,
                                            const int* __restrict__ col, const T* __restrict__ val, int beg, int end,
                                            int lane, int nvec, int r, int exact) {
  using Row = RowReg<T, VEC, GS, NIT>;
  constexpr int UN = (NIT == 1) ? 4 : 2;
  int e = beg;
  for (; e + UN <= end; e += UN) {
    int cj[UN]; T vj[UN]; Row xn[UN];
#pragma unroll
    for (int u = 0; u < UN; ++u) { cj[u] = __ldg(col + e + u); vj[u] = __ldg(val + e + u); }
#pragma unroll
    for (int u = 0; u < UN; ++u) xn[u].load(X + (int64_t)cj[u] * ld, lane, nvec, r, exact);
#pragma unroll
    for (int u = 0; u < UN; ++u) acc.axpy(vj[u], xn[u]);
  }
  for (; e < end; ++e) {
    Row xn; xn.load(X + (int64_t)__ldg(col + e) * ld, lane, nvec, r, exact);
    acc.axpy(__ldg(val + e), xn);
  }
}

// The adjoint pass is a chain of dependent gathers per row (pointers -> columns -> rows); it is bound by the number
// of warps that hide that latency, so its registers are capped for 6 blocks per SM (measured, min blocks 1 / 4 / 5 /
// 6 / 8: config 3 175 / 174 / 146 / 135 / 128 us, config 7 506 / 446 / 404 / 439 / 427 us, config 2 55 / 45 / 39 / 39 / 43 us)
#ifndef ALORA_ROWS_MINB
#define ALORA_ROWS_MINB 6
#endif
template <typename T, int VEC, int GS, int NIT, int MODE>
__global__ void __launch_bounds__(kBlock, (MODE == ROWS_ADJ && NIT <= 2) ? ALORA_ROWS_MINB : 1) k_rows(const RowArgs<T> a) {
  ALORA_GRID_DEP();
  using Row = RowReg<T, VEC, GS, NIT>;
  constexpr int GPB = kBlock / GS;
  constexpr int NST = (MODE == ROWS_LS_FUSED) ? 12 : 6;
  const int lane = threadIdx.x % GS, grp = threadIdx.x / GS;
  const unsigned gmask = group_mask<GS>();
  const int nvec = a.nvec, r = a.r, exact = a.exact;
  double st[NST];
#pragma unroll
  for (int s = 0; s < NST; ++s) st[s] = 0.0;

  for (int64_t pos = a.row_begin + (int64_t)blockIdx.x * GPB + grp; pos < a.n; pos += (int64_t)gridDim.x * GPB) {
    const int64_t row = a.perm ? (int64_t)__ldg(a.perm + pos) : pos;
    Row x; x.load(a.X + row * a.ld, lane, nvec, r, exact);
    const int cb = __ldg(a.c_rowptr + row), ce = __ldg(a.c_rowptr + row + 1);
    const T dc = __ldg(a.dC + row);

    if (MODE == ROWS_LS_FUSED) {
      Row d; d.load(a.X2 + row * a.ld, lane, nvec, r, exact);
      const T rr_l = x.dot(x), rd_l = x.dot(d), dd_l = d.dot(d);
      const double rr = group_sum<GS>((double)rr_l, gmask), rd = group_sum<GS>((double)rd_l, gmask),
                   dd = group_sum<GS>((double)dd_l, gmask);
      const int c = a.dcons ? __ldg(a.dcons + row) : (int)row;
      if (c >= 0 && lane == 0) {
        const double av = a.da ? (double)__ldg(a.da + row) : 1.0;
        const double q = av * rr - __ldg(a.b + c), q1 = 2.0 * av * rd, q2 = av * dd, yv = __ldg(a.y + c);
        st[LS_YQ] += yv * q; st[LS_YQ1] += yv * q1; st[LS_YQ2] += yv * q2;
        st[LS_QQ] += q * q; st[LS_QQ1] += q * q1; st[LS_QQ2] += q * q2;
        st[LS_Q11] += q1 * q1; st[LS_Q12] += q1 * q2; st[LS_Q22] += q2 * q2;
      }
      // <C, .> bilinear forms over the upper triangle (col > row), each off-diagonal pair once
      T sRR = T(0), sRD = T(0), sDD = T(0);
      for (int e = cb; e < ce; ++e) {
        const int k = __ldg(a.c_col + e);
        if (k > row) {
          const T cv = __ldg(a.c_val + e);
          Row xn, dn;
          xn.load(a.X + (int64_t)k * a.ld, lane, nvec, r, exact);
          dn.load(a.X2 + (int64_t)k * a.ld, lane, nvec, r, exact);
          sRR = fma(cv, x.dot(xn), sRR);
          sRD = fma(cv, x.dot(dn) + d.dot(xn), sRD);
          sDD = fma(cv, d.dot(dn), sDD);
        }
      }
      st[LS_CRR] += (double)dc * (double)rr_l + 2.0 * (double)sRR;
      st[LS_CRD] += (double)dc * (double)rd_l + (double)sRD;
      st[LS_CDD] += (double)dc * (double)dd_l + 2.0 * (double)sDD;
    } else {
      double coef = 0.0;  // weight of the row's own diagonal constraint times its coefficient
      if (MODE == ROWS_FUSED_EVAL) {
        const double nrm = group_sum<GS>((double)x.dot(x), gmask);
        const int c = a.dcons ? __ldg(a.dcons + row) : (int)row;
        if (c >= 0) {
          const double av = a.da ? (double)__ldg(a.da + row) : 1.0;
          const double z = av * nrm, q = z - __ldg(a.b + c), yv = __ldg(a.y + c), lam = yv - a.sigma * q;
          coef = lam * av;
          if (lane == 0) {
            if (a.z) a.z[c] = z;
            st[ES_YQ] += yv * q; st[ES_QQ] += q * q; st[ES_LZ] += lam * z;
          }
        }
      }
      // (C X)_row : diagonal + off-diagonal gathers
      Row acc; acc.zero(); acc.axpy(dc, x);
      if (MODE == ROWS_ADJ && a.nseg > 0 && ce - cb > kHeavyRow) {
        // heavy row: its off-diagonal C part was summed per segment by k_rows_seg and over the segments by k_heavy_sum
        int lo = 0, hi = a.nheavy - 1;
        while (lo < hi) { const int mid = (lo + hi) >> 1; if (__ldg(a.heavy_rows + mid) < (int)row) lo = mid + 1; else hi = mid; }
        const int s0 = __ldg(a.heavy_segptr + lo), s1 = __ldg(a.heavy_segptr + lo + 1);
        st[ES_CX] += (double)acc.dot(x);
        (void)s1;   // k_heavy_sum left the sum over the row's segments in its first segment's slot
        Row part; part.load(a.seg_out + (int64_t)s0 * (nvec * VEC), lane, nvec, r, exact);
        acc.axpy(T(1), part);
        if (lane == 0) st[ES_CX] += a.seg_cx[s0];
      } else {
        gather_axpy<T, VEC, GS, NIT>(acc, a.X, a.ld, a.c_col, a.c_val, cb, ce, lane, nvec, r, exact);
        st[ES_CX] += (double)acc.dot(x);
      }
      if (MODE == ROWS_ADJ) {
        if (a.diag_class) {
          const int c = a.dcons ? __ldg(a.dcons + row) : (int)row;
          if (c >= 0) coef = __ldg(a.w + c) * (a.da ? (double)__ldg(a.da + row) : 1.0);
        } else {
          const int ab = __ldg(a.a_rowptr + row), ae = __ldg(a.a_rowptr + row + 1);
          constexpr int UN = (NIT == 1) ? 4 : 2;
          int e = ab;
          for (; e + UN <= ae; e += UN) {
            int cj[UN]; T wj[UN]; Row xn[UN];
#pragma unroll
            for (int u = 0; u < UN; ++u) {
              cj[u] = __ldg(a.a_col + e + u);
              wj[u] = (T)(-__ldg(a.w + __ldg(a.a_cons + e + u)) * (double)__ldg(a.a_val + e + u));
            }
#pragma unroll
            for (int u = 0; u < UN; ++u) xn[u].load(a.X + (int64_t)cj[u] * a.ld, lane, nvec, r, exact);
#pragma unroll
            for (int u = 0; u < UN; ++u) acc.axpy(wj[u], xn[u]);
          }
          for (; e < ae; ++e) {
            Row xn; xn.load(a.X + (int64_t)__ldg(a.a_col + e) * a.ld, lane, nvec, r, exact);
            acc.axpy((T)(-__ldg(a.w + __ldg(a.a_cons + e)) * (double)__ldg(a.a_val + e)), xn);
          }
        }
        for (int p = 0; p < a.pC; ++p) {  // low-rank cost term: + U[row,p] * s_p (U^T X)_p
          const T up = __ldg(a.U + row * a.pC + p);
#pragma unroll
          for (int it = 0; it < NIT; ++it) {
            const int vi = lane + it * GS;
            if (vi < nvec) {
#pragma unroll
              for (int i = 0; i < VEC; ++i) {
                const int cidx = vi * VEC + i;
                if (cidx < r) acc.p[it].v[i] = fma(up, (T)__ldg(a.Ts + p * r + cidx), acc.p[it].v[i]);
              }
            }
          }
        }
      }
      acc.axpy((T)(-coef), x);
      const T sc = (T)a.scale;
#pragma unroll
      for (int it = 0; it < NIT; ++it)
#pragma unroll
        for (int i = 0; i < VEC; ++i) acc.p[it].v[i] *= sc;
      st[ES_GG] += (double)acc.dot(acc);
      st[ES_GR] += (double)acc.dot(x);
      if (a.Out) acc.store(a.Out + row * a.ld, lane, nvec, r, exact);
    }
  }
  block_reduce_store<NST>(st, a.partials + (int64_t)blockIdx.x * kNStat);
  finish_partials(a.fin);
}

// ---------------------------------------------------------------------------------------------
// Weighted-adjoint SpMM for LONG rows (general class, tens of entries per row): one WARP per row, the 32 lanes
// split as PL pack lanes x EL = 32 / PL entry lanes.  Entry lane el walks entries el, el + EL, ... of the row's C
// list and of its constraint list, so a row has EL independent gather chains instead of one; the partial rows are
// added across the entry lanes with shuffles at the end.  <C,XX^T> needs the C part alone: every lane keeps its own
// scalar sum of c_e <X_k, X_row> over the C entries it handled (no extra reduction).  ROWS_ADJ semantics.
template <typename T, int VEC, int PL, int NIT>
__global__ void __launch_bounds__(kBlock) k_rows_ep(const RowArgs<T> a) {
  ALORA_GRID_DEP();
  using Row = RowReg<T, VEC, PL, NIT>;
  constexpr int EL = 32 / PL, WPB = kBlock / 32, NST = 6;
  const int lane32 = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int pl = lane32 % PL, el = lane32 / PL;
  const int nvec = a.nvec, r = a.r, exact = a.exact;
  const T sc = (T)a.scale;
  double st[NST];
#pragma unroll
  for (int s = 0; s < NST; ++s) st[s] = 0.0;
  for (int64_t row = (int64_t)blockIdx.x * WPB + warp; row < a.n; row += (int64_t)gridDim.x * WPB) {
    Row x; x.load(a.X + row * a.ld, pl, nvec, r, exact);
    Row acc; acc.zero();
    T cxl = T(0);
    const int cb = __ldg(a.c_rowptr + row), ce = __ldg(a.c_rowptr + row + 1);
    if (a.nseg > 0 && ce - cb > kHeavyRow) {
      // heavy row: its C part was summed per segment by k_rows_seg and over the segments by k_heavy_sum
      int lo = 0, hi = a.nheavy - 1;
      while (lo < hi) { const int mid = (lo + hi) >> 1; if (__ldg(a.heavy_rows + mid) < (int)row) lo = mid + 1; else hi = mid; }
      const int s0 = __ldg(a.heavy_segptr + lo), s1 = __ldg(a.heavy_segptr + lo + 1);
      (void)s1;   // k_heavy_sum left the sum over the row's segments in its first segment's slot
      if (el == 0) {
        Row part; part.load(a.seg_out + (int64_t)s0 * (nvec * VEC), pl, nvec, r, exact);
        acc.axpy(T(1), part);
        if (pl == 0) st[ES_CX] += a.seg_cx[s0];
      }
    } else {
#pragma unroll 2
      for (int e = cb + el; e < ce; e += EL) {
        const int k = __ldg(a.c_col + e);
        const T v = __ldg(a.c_val + e);
        Row xn; xn.load(a.X + (int64_t)k * a.ld, pl, nvec, r, exact);
        acc.axpy(v, xn);
        cxl = fma(v, xn.dot(x), cxl);
      }
    }
    double coef = 0.0;
    if (a.diag_class) {
      const int c = a.dcons ? __ldg(a.dcons + row) : (int)row;
      if (c >= 0) coef = __ldg(a.w + c) * (a.da ? (double)__ldg(a.da + row) : 1.0);
    } else {
      const int ab = __ldg(a.a_rowptr + row), ae = __ldg(a.a_rowptr + row + 1);
#pragma unroll 2
      for (int e = ab + el; e < ae; e += EL) {
        const int k = __ldg(a.a_col + e);
        const T wv = (T)(-__ldg(a.w + __ldg(a.a_cons + e)) * (double)__ldg(a.a_val + e));
        Row xn; xn.load(a.X + (int64_t)k * a.ld, pl, nvec, r, exact);
        acc.axpy(wv, xn);
      }
    }
#pragma unroll
    for (int off = PL; off < 32; off <<= 1)
#pragma unroll
      for (int it = 0; it < NIT; ++it)
#pragma unroll
        for (int i = 0; i < VEC; ++i) acc.p[it].v[i] += __shfl_xor_sync(0xffffffffu, acc.p[it].v[i], off);
    // every entry lane now holds the whole row; entry lane 0 finishes it
    const T dc = __ldg(a.dC + row);
    if (el == 0) cxl = fma(dc, x.dot(x), cxl);
    acc.axpy(dc, x);
    for (int p = 0; p < a.pC; ++p) {  // low-rank cost term: + U[row,p] * s_p (U^T X)_p
      const T up = __ldg(a.U + row * a.pC + p);
#pragma unroll
      for (int it = 0; it < NIT; ++it) {
        const int vi = pl + it * PL;
        if (vi < nvec) {
#pragma unroll
          for (int i = 0; i < VEC; ++i) {
            const int cidx = vi * VEC + i;
            if (cidx < r) acc.p[it].v[i] = fma(up, (T)__ldg(a.Ts + p * r + cidx), acc.p[it].v[i]);
          }
        }
      }
    }
    acc.axpy((T)(-coef), x);
#pragma unroll
    for (int it = 0; it < NIT; ++it)
#pragma unroll
      for (int i = 0; i < VEC; ++i) acc.p[it].v[i] *= sc;
    st[ES_CX] += (double)cxl;
    if (el == 0) {
      st[ES_GG] += (double)acc.dot(acc);
      st[ES_GR] += (double)acc.dot(x);
      if (a.Out) acc.store(a.Out + row * a.ld, pl, nvec, r, exact);
    }
  }
  block_reduce_store<NST>(st, a.partials + (int64_t)blockIdx.x * kNStat);
  finish_partials(a.fin);
}

// ---------------------------------------------------------------------------------------------
// Weighted-adjoint SpMM of the general class, cooperative warp per row ("cw").  The thread-per-item kernels of this
// path are bound by the L1 request pipeline, not by bytes (profiles/r2b_README.md: k_cons1 runs at 85 % of the L1
// throughput with 9 % of the issue slots used) -- a request is one 128-byte line touched by one warp instruction.  So
//   * the entry metadata of a row (column, value, constraint id) is read 32 entries at a time, one entry per lane
//     (coalesced: one request per array per 32 entries instead of one per entry), the weight lambda[cons] is
//     gathered by the lane that owns the entry, and the lane forms the entry's coefficient c_e or -lambda_i a_e;
//   * the neighbour rows are then gathered EL = 32 / PL entries per instruction: PL (a power of two >= the packs of
//     a row) consecutive lanes take the consecutive packs of one row, column and coefficient arriving by shuffle --
//     one request per gathered row;
//   * every lane accumulates one pack; the EL partial rows are added by a butterfly once per row.
// ROWS_ADJ semantics (Out = scale * (C - sum_i w_i A_i) X, <C,XX^T>, |Out|^2, <Out,X>), nvec <= PL.
template <typename T, int VEC, int PL, int UNR>
__global__ void __launch_bounds__(kBlock) k_rows_cw(const RowArgs<T> a) {
  ALORA_GRID_DEP();
  constexpr int WPB = kBlock / 32, NST = 6, EL = 32 / PL;
  using P = Pack<T, VEC>;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int nvec = a.nvec, r = a.r;
  const int pl = lane & (PL - 1), el = lane / PL;
  const bool pok = pl < nvec;                    // this lane owns a pack of the row
  const bool tailmask = VEC > 1 && !a.exact && pl == nvec - 1;
  const int64_t ld = a.ld;
  const uint32_t ld32 = (uint32_t)a.ld;          // the host selects this kernel only when n * ld < 2^32 elements
  const int plc = min(pl, nvec - 1);             // lanes beyond the row read its last pack (same request) and drop it
  const T* const Xp = a.X + plc * VEC;           // lane's pack of row 0
  const T sc = (T)a.scale;
  double st[NST];
#pragma unroll
  for (int s = 0; s < NST; ++s) st[s] = 0.0;
  auto zero = [] { P z;
#pragma unroll
    for (int i = 0; i < VEC; ++i) z.v[i] = T(0);
    return z; };
  // p points at the lane's pack.  The load is unconditional (a branch around it costs a convergence barrier per load);
  // lanes that own no pack and the elements beyond r (partial last pack) are zeroed by selects.
  const int nkeep = !pok ? 0 : (tailmask ? r - pl * VEC : VEC);
  auto load_pack = [&](const T* p) {
    P v = ldg_pack<T, VEC>(p);
#pragma unroll
    for (int i = 0; i < VEC; ++i) v.v[i] = i < nkeep ? v.v[i] : T(0);
    return v;
  };
  // the 32 (column, coefficient) pairs of a batch pass from the lanes that loaded them to the lanes that use them
  // through a warp-private piece of shared memory (a shuffle inside this data-dependent loop would cost a
  // convergence barrier each)
  __shared__ int s_col[WPB][32];
  __shared__ T s_cf[WPB][32];
  int* const colS = s_col[warp]; T* const cfS = s_cf[warp];
  for (int64_t pos = (int64_t)blockIdx.x * WPB + warp; pos < a.n; pos += (int64_t)gridDim.x * WPB) {
    const int64_t row = a.perm ? (int64_t)__ldg(a.perm + pos) : pos;
    const P x = load_pack(Xp + row * ld);
    P acc = zero();
    // one list of entries [beg, end): coefficients val[e] (cons == nullptr) or -w[cons[e]] * val[e]
    auto walk = [&](const int* __restrict__ col, const T* __restrict__ val, const int* __restrict__ cons, int beg, int end) {
      for (int base = beg; base < end; base += 32) {
        const int e = base + lane;
        int col_l = (int)row; T cf_l = T(0);       // padding entries: the row itself with coefficient 0
        if (e < end) {
          col_l = __ldg(col + e);
          const T v = __ldg(val + e);
          cf_l = cons ? (T)(-__ldg(a.w + __ldg(cons + e)) * (double)v) : v;
        }
        colS[lane] = col_l; cfS[lane] = cf_l;
        __syncwarp();
        const int cnt = min(32, end - base);
        for (int j = el; j < cnt; j += EL * UNR) {
          P pk[UNR]; T cf[UNR];
#pragma unroll
          for (int u = 0; u < UNR; ++u) {
            const int src = j + u * EL;          // < 32: EL * UNR <= 32 and j - el is a multiple of EL * UNR
            cf[u] = cfS[src];
            pk[u] = load_pack(Xp + (uint32_t)colS[src] * ld32);   // 32-bit element offset: two instructions instead of seven
          }
#pragma unroll
          for (int u = 0; u < UNR; ++u)
#pragma unroll
            for (int i = 0; i < VEC; ++i) acc.v[i] = fma(cf[u], pk[u].v[i], acc.v[i]);
        }
        __syncwarp();
      }
    };
    const int cb = __ldg(a.c_rowptr + row), ce = __ldg(a.c_rowptr + row + 1);
    if (a.nseg > 0 && ce - cb > kHeavyRow) {
      // heavy row: its C part was summed per segment by k_rows_seg and over the segments by k_heavy_sum
      int lo = 0, hi = a.nheavy - 1;
      while (lo < hi) { const int mid = (lo + hi) >> 1; if (__ldg(a.heavy_rows + mid) < (int)row) lo = mid + 1; else hi = mid; }
      const int s0 = __ldg(a.heavy_segptr + lo), s1 = __ldg(a.heavy_segptr + lo + 1);
      (void)s1;   // k_heavy_sum left the sum over the row's segments in its first segment's slot
      if (el == 0) {
        const P part = load_pack(a.seg_out + (int64_t)s0 * (nvec * VEC) + plc * VEC);
#pragma unroll
        for (int i = 0; i < VEC; ++i) acc.v[i] += part.v[i];
        if (lane == 0) st[ES_CX] += a.seg_cx[s0];
      }
    } else {
      walk(a.c_col, a.c_val, nullptr, cb, ce);
      T cxl = T(0);   // lane-partial <(C_offdiag X)_row, X_row>: every lane holds part of the row sum of its pack
#pragma unroll
      for (int i = 0; i < VEC; ++i) cxl = fma(acc.v[i], x.v[i], cxl);
      st[ES_CX] += (double)cxl;
    }
    double coef = 0.0;
    if (a.diag_class) {
      const int c = a.dcons ? __ldg(a.dcons + row) : (int)row;
      if (c >= 0) coef = __ldg(a.w + c) * (a.da ? (double)__ldg(a.da + row) : 1.0);
    } else {
      walk(a.a_col, a.a_val, a.a_cons, __ldg(a.a_rowptr + row), __ldg(a.a_rowptr + row + 1));
    }
    // add the EL partial rows (lanes with the same pl): butterfly over the entry-lane bits
#pragma unroll
    for (int off = PL; off < 32; off <<= 1)
#pragma unroll
      for (int i = 0; i < VEC; ++i) acc.v[i] += __shfl_xor_sync(0xffffffffu, acc.v[i], off);
    if (el == 0 && pok) {
      const T dc = __ldg(a.dC + row);
      T xx = T(0);
#pragma unroll
      for (int i = 0; i < VEC; ++i) { xx = fma(x.v[i], x.v[i], xx); acc.v[i] = fma(dc, x.v[i], acc.v[i]); }
      st[ES_CX] += (double)(dc * xx);
      for (int p = 0; p < a.pC; ++p) {  // low-rank cost term: + U[row,p] * s_p (U^T X)_p
        const T up = __ldg(a.U + row * a.pC + p);
#pragma unroll
        for (int i = 0; i < VEC; ++i) {
          const int cidx = pl * VEC + i;
          if (cidx < r) acc.v[i] = fma(up, (T)__ldg(a.Ts + p * r + cidx), acc.v[i]);
        }
      }
      T gg = T(0), gr = T(0);
#pragma unroll
      for (int i = 0; i < VEC; ++i) {
        acc.v[i] = fma((T)(-coef), x.v[i], acc.v[i]) * sc;
        gg = fma(acc.v[i], acc.v[i], gg); gr = fma(acc.v[i], x.v[i], gr);
      }
      st[ES_GG] += (double)gg; st[ES_GR] += (double)gr;
      if (a.Out) {
        T* o = a.Out + row * ld + pl * VEC;
        if (tailmask) {
#pragma unroll
          for (int i = 0; i < VEC; ++i) if (pl * VEC + i < r) o[i] = acc.v[i];
        } else {
          st_pack<T, VEC>(o, acc);
        }
      }
    }
  }
  block_reduce_store<NST>(st, a.partials + (int64_t)blockIdx.x * kNStat);
  finish_partials(a.fin);
}

// Segment pass of k_rows_ep: a warp per segment (<= kHeavyRow consecutive C entries of a heavy row) leaves
// sum_e c_e X_{k_e} in seg_out[s][0..r) and sum_e c_e <X_{k_e}, X_row> in seg_cx[s].
template <typename T, int VEC, int PL, int NIT>
__global__ void __launch_bounds__(kBlock) k_rows_seg(const RowArgs<T> a) {
  ALORA_GRID_DEP();
  using Row = RowReg<T, VEC, PL, NIT>;
  constexpr int EL = 32 / PL, WPB = kBlock / 32;
  const int lane32 = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int pl = lane32 % PL, el = lane32 / PL;
  const int nvec = a.nvec, r = a.r, exact = a.exact;
  for (int sg = blockIdx.x * WPB + warp; sg < a.nseg; sg += gridDim.x * WPB) {
    const int64_t row = __ldg(a.seg_row + sg);
    Row x; x.load(a.X + row * a.ld, pl, nvec, r, exact);
    Row acc; acc.zero();
    T cxl = T(0);
    const int eb = __ldg(a.seg_beg + sg), ee = __ldg(a.seg_end + sg);
#pragma unroll 2
    for (int e = eb + el; e < ee; e += EL) {
      const int k = __ldg(a.c_col + e);
      const T v = __ldg(a.c_val + e);
      Row xn; xn.load(a.X + (int64_t)k * a.ld, pl, nvec, r, exact);
      acc.axpy(v, xn);
      cxl = fma(v, xn.dot(x), cxl);
    }
#pragma unroll
    for (int off = PL; off < 32; off <<= 1)
#pragma unroll
      for (int it = 0; it < NIT; ++it)
#pragma unroll
        for (int i = 0; i < VEC; ++i) acc.p[it].v[i] += __shfl_xor_sync(0xffffffffu, acc.p[it].v[i], off);
    const double cx = warp_sum((double)cxl);
    if (el == 0) acc.store(a.seg_out + (int64_t)sg * (nvec * VEC), pl, nvec, r, exact);
    if (lane32 == 0) a.seg_cx[sg] = cx;
  }
}

// Second level of the heavy-row sums: a warp per heavy row adds the partial rows (and the <C X, X> parts) of the row's
// segments in a fixed order and leaves the total in the FIRST segment's slot, which is all the row kernels then read.
// Before, the group that owned the row added its segments one dependent load at a time -- 308 segments for the
// largest row of config 7 -- and the whole grid waited for that group (ncu: the SMs were active for 42 % of the
// adjoint kernel's duration).  Lanes: PW = smallest power of two >= P elements of a partial row (capped at 32) take the
// elements, the 32 / PW lane groups take every (32 / PW)-th segment; the groups' sums are then added in group order.
template <typename T>
__global__ void __launch_bounds__(kBlock) k_heavy_sum(int nheavy, const int* __restrict__ heavy_segptr, T* seg_out, double* seg_cx, int P) {
  ALORA_GRID_DEP();
  constexpr int WPB = kBlock / 32;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int PW = 1; while (PW < P && PW < 32) PW <<= 1;
  const int NG = 32 / PW, g = lane / PW, el0 = lane % PW;
  for (int h = blockIdx.x * WPB + warp; h < nheavy; h += gridDim.x * WPB) {
    const int s0 = __ldg(heavy_segptr + h), s1 = __ldg(heavy_segptr + h + 1);
    double cx = 0.0;
    for (int sg = s0 + lane; sg < s1; sg += 32) cx += __ldcg(seg_cx + sg);
    cx = warp_sum(cx);
    for (int eb = 0; eb < P; eb += PW) {   // one pass unless a partial row has more than 32 elements
      const int el = eb + el0;
      T acc = T(0);
      if (el < P) {
        int sg = s0 + g;
        for (; sg + 7 * NG < s1; sg += 8 * NG) {   // eight loads in flight, added in segment order
          T v[8];
#pragma unroll
          for (int u = 0; u < 8; ++u) v[u] = __ldcg(seg_out + (int64_t)(sg + u * NG) * P + el);
#pragma unroll
          for (int u = 0; u < 8; ++u) acc += v[u];
        }
        for (; sg < s1; sg += NG) acc += __ldcg(seg_out + (int64_t)sg * P + el);
      }
      T tot = T(0);
      for (int q = 0; q < NG; ++q) tot += __shfl_sync(0xffffffffu, acc, q * PW + el0);   // groups in order
      __syncwarp();   // every lane has read its segments before the first slot is overwritten
      if (g == 0 && el < P) seg_out[(int64_t)s0 * P + el] = tot;
    }
    if (lane == 0) seg_cx[s0] = cx;
  }
}

// ---------------------------------------------------------------------------------------------
// Forward (SDDMM-style) evaluator.  One entry e = (j, k, a), j <= k, contributes
//   w a <X_j, X_k>                 with w = 1 (j == k) or 2 (j < k)            -> z
//   w a (<X_j,D_k> + <D_j,X_k>)    (= <A, XD^T + DX^T> restricted to the entry)  -> q1
//   w a <D_j, D_k>                                                               -> q2
template <typename T, int VEC, int GS, int NIT, int MODE>
__device__ __forceinline__ void cons_entry(const ConsArgs<T>& a, int64_t e, int lane, T& s0, T& s1, T& s2) {
  using Row = RowReg<T, VEC, GS, NIT>;
  const int j = __ldg(a.e_row + e), k = __ldg(a.e_col + e);
  T av = __ldg(a.e_val + e);
  Row xj, xk;
  xj.load(a.X + (int64_t)j * a.ld, lane, a.nvec, a.r, a.exact);
  if (j != k) { av += av; xk.load(a.X + (int64_t)k * a.ld, lane, a.nvec, a.r, a.exact); } else { xk = xj; }
  s0 = fma(av, xj.dot(xk), s0);
  if (MODE == CONS_LS) {
    Row dj, dk;
    dj.load(a.X2 + (int64_t)j * a.ld, lane, a.nvec, a.r, a.exact);
    if (j != k) dk.load(a.X2 + (int64_t)k * a.ld, lane, a.nvec, a.r, a.exact); else dk = dj;
    s1 = fma(av, xj.dot(dk) + dj.dot(xk), s1);
    s2 = fma(av, dj.dot(dk), s2);
  }
}

// per-constraint finalisation (a2): q = z - b, lambda = y - sigma q, scalar sums
template <int MODE>
__device__ __forceinline__ void cons_finish(double* st, int64_t i, double z, double q1, double q2,
                                            const double* y, const double* b, double sigma, double* zout,
                                            double* lam) {
  const double q = z - __ldg(b + i), yv = __ldg(y + i);
  if (MODE == CONS_EVAL) {
    const double l = yv - sigma * q;
    zout[i] = z; lam[i] = l;
    st[ES_YQ] += yv * q; st[ES_QQ] += q * q; st[ES_LZ] += l * z;
  } else {
    st[LS_YQ] += yv * q; st[LS_YQ1] += yv * q1; st[LS_YQ2] += yv * q2;
    st[LS_QQ] += q * q; st[LS_QQ1] += q * q1; st[LS_QQ2] += q * q2;
    st[LS_Q11] += q1 * q1; st[LS_Q12] += q1 * q2; st[LS_Q22] += q2 * q2;
  }
}

template <typename T, int VEC, int GS, int NIT, int MODE>
__global__ void __launch_bounds__(kBlock) k_cons(const ConsArgs<T> a) {
  ALORA_GRID_DEP();
  constexpr int GPB = kBlock / GS;
  constexpr int NST = (MODE == CONS_LS) ? 12 : 6;
  const int lane = threadIdx.x % GS, grp = threadIdx.x / GS;
  const unsigned gmask = group_mask<GS>();
  double st[NST];
#pragma unroll
  for (int s = 0; s < NST; ++s) st[s] = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * GPB + grp; i < a.m; i += (int64_t)gridDim.x * GPB) {
    const int64_t e0 = __ldg(a.ptr + i), e1 = __ldg(a.ptr + i + 1);
    if (e1 - e0 > kLongThreshold) continue;  // long constraints: k_cons_chunk + k_long_finish
    T s0 = T(0), s1 = T(0), s2 = T(0);
#pragma unroll 4
    for (int64_t e = e0; e < e1; ++e) cons_entry<T, VEC, GS, NIT, MODE>(a, e, lane, s0, s1, s2);
    const double z = group_sum<GS>((double)s0, gmask);
    double q1 = 0.0, q2 = 0.0;
    if (MODE == CONS_LS) { q1 = group_sum<GS>((double)s1, gmask); q2 = group_sum<GS>((double)s2, gmask); }
    if (lane == 0) cons_finish<MODE>(st, i, z, q1, q2, a.y, a.b, a.sigma, a.z, a.lam);
  }
  block_reduce_store<NST>(st, a.partials + (int64_t)blockIdx.x * kNStat);
  finish_partials(a.fin);
}

// Forward evaluator with one THREAD per constraint, for constraints with few stored entries (SINGLE: exactly one
// each -- matrix completion, the edge constraints of theta; otherwise a short list via ptr -- random sparse
// constraints): a warp instruction serves 32 constraints instead of 32 / GS.  The constraint streams (entries, y, b
// in; z, lambda out) are coalesced; the rows are gathered pack by pack (R is small and L2-resident in these
// workloads).  Constraints with more than kLongThreshold entries are skipped (chunk kernels), as in k_cons.  Same
// sums as k_cons.
template <typename T, int VEC, int MODE, bool SINGLE>
__global__ void __launch_bounds__(kBlock) k_cons1(const ConsArgs<T> a) {
  ALORA_GRID_DEP();
  constexpr int NST = (MODE == CONS_LS) ? 12 : 6;
  double st[NST];
#pragma unroll
  for (int s = 0; s < NST; ++s) st[s] = 0.0;
  const int nvec = a.nvec, r = a.r;
  for (int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x; i < a.m; i += (int64_t)gridDim.x * kBlock) {
    const int64_t e0 = SINGLE ? i : __ldg(a.ptr + i), e1 = SINGLE ? i + 1 : __ldg(a.ptr + i + 1);
    if (!SINGLE && e1 - e0 > kLongThreshold) continue;
    T t0 = T(0), t1 = T(0), t2 = T(0);
    for (int64_t e = e0; e < e1; ++e) {
      const int j = __ldg(a.e_row + e), k = __ldg(a.e_col + e);
      T av = __ldg(a.e_val + e);
      if (j != k) av += av;
      const T* xj = a.X + (int64_t)j * a.ld; const T* xk = a.X + (int64_t)k * a.ld;
      T s0 = T(0), s1 = T(0), s2 = T(0);
      for (int v = 0; v < nvec; ++v) {
        Pack<T, VEC> pj = ldg_pack<T, VEC>(xj + v * VEC), pk = ldg_pack<T, VEC>(xk + v * VEC);
        Pack<T, VEC> dj, dk;
        if (MODE == CONS_LS) { dj = ldg_pack<T, VEC>(a.X2 + (int64_t)j * a.ld + v * VEC); dk = ldg_pack<T, VEC>(a.X2 + (int64_t)k * a.ld + v * VEC); }
#pragma unroll
        for (int q = 0; q < VEC; ++q) {
          if (VEC > 1 && v * VEC + q >= r) break;   // partial last pack
          s0 = fma(pj.v[q], pk.v[q], s0);
          if (MODE == CONS_LS) { s1 = fma(pj.v[q], dk.v[q], fma(dj.v[q], pk.v[q], s1)); s2 = fma(dj.v[q], dk.v[q], s2); }
        }
      }
      t0 = fma(av, s0, t0); t1 = fma(av, s1, t1); t2 = fma(av, s2, t2);
    }
    cons_finish<MODE>(st, i, (double)t0, (double)t1, (double)t2, a.y, a.b, a.sigma, a.z, a.lam);
  }
  block_reduce_store<NST>(st, a.partials + (int64_t)blockIdx.x * kNStat);
  finish_partials(a.fin);
}

// ---------------------------------------------------------------------------------------------
// Cooperative forward evaluator ("cw", same idea as k_rows_cw): a warp takes 32 consecutive forward entries, reads
// their (row, col, value) one entry per lane (coalesced), then gathers the two rows of EL = 32 / PL entries per
// instruction with PL consecutive lanes on the consecutive packs of a row (one request per row instead of one per
// pack), forms the lane-partial dot products, adds them over the PL lanes of an entry by a butterfly, and the entry's
// first lane scales by w a.  SINGLE (every constraint is one entry): that lane finishes the constraint in place.
// Otherwise the per-entry sums go to e_out and k_cons_fin / k_long_fin_e add them per constraint in a fixed order.
// Entries beyond nf_A are C's sym-upper list (line search): <C,RR^T>, <C,RD^T>, <C,DD^T> straight into the stats.
template <typename T, int VEC, int PL, int MODE, bool SINGLE, int UNR>
__global__ void __launch_bounds__(kBlock) k_ent_cw(const ConsArgs<T> a) {
  ALORA_GRID_DEP();
  constexpr int WPB = kBlock / 32, NST = (MODE == CONS_LS) ? 12 : 6, K = (MODE == CONS_LS) ? 3 : 1, EL = 32 / PL;
  constexpr bool LS = (MODE == CONS_LS);
  using P = Pack<T, VEC>;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int nvec = a.nvec, r = a.r;
  const int pl = lane & (PL - 1), el = lane / PL;
  const bool pok = pl < nvec;
  const bool tailmask = VEC > 1 && !a.exact && pl == nvec - 1;
  const uint32_t ld32 = (uint32_t)a.ld;          // the host selects this kernel only when n * ld < 2^32 elements
  const int plc = min(pl, nvec - 1);
  const T* const Xp = a.X + plc * VEC;
  const T* const Dp = LS ? a.X2 + plc * VEC : nullptr;
  double st[NST];
#pragma unroll
  for (int s = 0; s < NST; ++s) st[s] = 0.0;
  auto zero = [] { P z;
#pragma unroll
    for (int i = 0; i < VEC; ++i) z.v[i] = T(0);
    return z; };
  const int nkeep = !pok ? 0 : (tailmask ? r - pl * VEC : VEC);   // elements of the lane's pack that exist
  auto load_pack = [&](const T* p) {   // unconditional load, lanes without a pack / elements beyond r zeroed by selects
    P v = ldg_pack<T, VEC>(p);
#pragma unroll
    for (int i = 0; i < VEC; ++i) v.v[i] = i < nkeep ? v.v[i] : T(0);
    return v;
  };
  auto dotp = [](const P& x, const P& y) { T t = T(0);
#pragma unroll
    for (int i = 0; i < VEC; ++i) t = fma(x.v[i], y.v[i], t);
    return t; };
  auto seg = [](T v) {   // sum over the PL lanes of an entry (every lane gets it)
#pragma unroll
    for (int off = PL / 2; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    return v; };
  // uniform constraints (a.npc > 1 entries each, npc | 32): the entry sums of a batch meet in shared memory and the
  // first 32 / npc lanes finish the batch's constraints -- no e_out, no second kernel
  __shared__ T s_ev[SINGLE ? 1 : WPB][SINGLE ? 1 : 32 * K];
  T* const evS = s_ev[SINGLE ? 0 : warp];
  const int npc = SINGLE ? 1 : a.npc;
  // Every loop below has a block-uniform or compile-time trip count, so the shuffles need no convergence barriers:
  // a block takes WPB batches at a time, warps whose batch starts beyond the list run on padding entries (row 0 with
  // itself, coefficient 0) and write nothing.
  for (int64_t cbk = blockIdx.x; cbk * (WPB * 32) < a.nent; cbk += gridDim.x) {
    const int64_t base = (cbk * WPB + warp) * 32;
    const int64_t e = base + lane;
    int jr = 0, kc = 0; T av = T(0);
    if (e < a.nent) { jr = __ldg(a.e_row + e); kc = __ldg(a.e_col + e); av = __ldg(a.e_val + e); if (jr != kc) av += av; }
    // slots [0, lim_A) of the batch are constraint entries, [lim_A, lim_ent) entries of C's list (32-bit compares below)
    const int lim_ent = (int)max((int64_t)0, min((int64_t)32, a.nent - base));
    const int lim_A = (int)max((int64_t)0, min((int64_t)32, a.nf_A - base));
#pragma unroll
    for (int j = 0; j < 32; j += EL * UNR) {
      P xj[UNR], xk[UNR], dj[UNR], dk[UNR];
      T au[UNR];
#pragma unroll
      for (int u = 0; u < UNR; ++u) {
        const int src = j + u * EL + el;
        const int ju = __shfl_sync(0xffffffffu, jr, src), ku = __shfl_sync(0xffffffffu, kc, src);
        au[u] = __shfl_sync(0xffffffffu, av, src);
        const uint32_t oj = (uint32_t)ju * ld32, ok = (uint32_t)ku * ld32;   // 32-bit element offsets
        xj[u] = load_pack(Xp + oj);
        xk[u] = ku != ju ? load_pack(Xp + ok) : xj[u];
        if (LS) {
          dj[u] = load_pack(Dp + oj);
          dk[u] = ku != ju ? load_pack(Dp + ok) : dj[u];
        }
      }
#pragma unroll
      for (int u = 0; u < UNR; ++u) {
        const T s0 = seg(dotp(xj[u], xk[u]));
        T s1 = T(0), s2 = T(0);
        if (LS) { s1 = seg(dotp(xj[u], dk[u]) + dotp(dj[u], xk[u])); s2 = seg(dotp(dj[u], dk[u])); }
        const int slot = j + u * EL + el;
        const int64_t ei = base + slot;
        if (pl == 0 && slot < lim_ent) {
          const T v0 = au[u] * s0, v1 = au[u] * s1, v2 = au[u] * s2;
          if (slot < lim_A) {
            if (SINGLE) {
              cons_finish<MODE>(st, ei, (double)v0, (double)v1, (double)v2, a.y, a.b, a.sigma, a.z, a.lam);
            } else if (npc > 1) {
              const int sl = slot * K;
              evS[sl] = v0;
              if (LS) { evS[sl + 1] = v1; evS[sl + 2] = v2; }
            } else {
              a.e_out[ei * K] = v0;
              if (LS) { a.e_out[ei * K + 1] = v1; a.e_out[ei * K + 2] = v2; }
            }
          } else if (LS) {   // C's sym-upper list: the entry sums are <C,RR^T>, <C,RD^T + DR^T>, <C,DD^T> restricted to the entry
            st[LS_CRR] += (double)v0; st[LS_CRD] += 0.5 * (double)v1; st[LS_CDD] += (double)v2;
          }
        }
      }
    }
    if (!SINGLE && npc > 1) {   // block-uniform condition
      __syncwarp();
      const int64_t ci = base / npc + lane;          // base is a multiple of 32, hence of npc
      if (lane < 32 / npc && ci < a.m) {
        double t0 = 0.0, t1 = 0.0, t2 = 0.0;
        for (int t = 0; t < npc; ++t) {
          const int sl = (lane * npc + t) * K;
          t0 += (double)evS[sl];
          if (LS) { t1 += (double)evS[sl + 1]; t2 += (double)evS[sl + 2]; }
        }
        cons_finish<MODE>(st, ci, t0, t1, t2, a.y, a.b, a.sigma, a.z, a.lam);
      }
      __syncwarp();
    }
  }
  block_reduce_store<NST>(st, a.partials + (int64_t)blockIdx.x * kNStat);
  finish_partials(a.fin);
}

// per-constraint sums of the entry results of k_ent_cw (constraints with at most kLongThreshold entries), a thread
// per constraint, entries added in list order, then the per-constraint finish (a2)
template <typename T, int MODE>
__global__ void __launch_bounds__(kBlock) k_cons_fin(const ConsArgs<T> a) {
  ALORA_GRID_DEP();
  constexpr int NST = (MODE == CONS_LS) ? 12 : 6, K = (MODE == CONS_LS) ? 3 : 1;
  double st[NST];
#pragma unroll
  for (int s = 0; s < NST; ++s) st[s] = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x; i < a.m; i += (int64_t)gridDim.x * kBlock) {
    const int64_t e0 = __ldg(a.ptr + i), e1 = __ldg(a.ptr + i + 1);
    if (e1 - e0 > kLongThreshold) continue;
    double t0 = 0.0, t1 = 0.0, t2 = 0.0;
    for (int64_t e = e0; e < e1; ++e) {
      t0 += (double)a.e_out[e * K];
      if (MODE == CONS_LS) { t1 += (double)a.e_out[e * K + 1]; t2 += (double)a.e_out[e * K + 2]; }
    }
    cons_finish<MODE>(st, i, t0, t1, t2, a.y, a.b, a.sigma, a.z, a.lam);
  }
  block_reduce_store<NST>(st, a.part_chunk + (int64_t)blockIdx.x * kNStat);
  finish_partials(a.fin);
}

// the same for one long constraint per block of kLongFinThreads threads: thread t adds entries t, t + 1024, ... in order,
// then an ordered block sum (one block per constraint: the trace row of the theta SDP has n entries, and with 256
// threads this kernel took 14 / 38 us on config 2 -- ten dependent round trips; 1024 threads make it three)
constexpr int kLongFinThreads = 1024;
template <typename T, int MODE>
__global__ void __launch_bounds__(kLongFinThreads) k_long_fin_e(const ConsArgs<T> a, double* part_long) {
  ALORA_GRID_DEP();
  constexpr int K = (MODE == CONS_LS) ? 3 : 1, BT = kLongFinThreads;
  __shared__ double sm[3][BT / 32];
  const int slot = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int64_t i = a.long_cons[slot], e0 = a.ptr[i], e1 = a.ptr[i + 1];
  double v[3] = {0.0, 0.0, 0.0};
  constexpr int U = 8;   // loads in flight per thread (the sums stay in entry order)
  for (int64_t eb = e0 + threadIdx.x; eb < e1; eb += (int64_t)BT * U) {
    T t[U][K];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t e = eb + (int64_t)u * BT;
#pragma unroll
      for (int k = 0; k < K; ++k) t[u][k] = e < e1 ? __ldcg(a.e_out + e * K + k) : T(0);
    }
#pragma unroll
    for (int u = 0; u < U; ++u)
#pragma unroll
      for (int k = 0; k < K; ++k) v[k] += (double)t[u][k];
  }
  for (int k = 0; k < 3; ++k) { const double t = warp_sum(v[k]); if (lane == 0) sm[k][warp] = t; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double t[3] = {0.0, 0.0, 0.0};
    for (int k = 0; k < 3; ++k) for (int wv = 0; wv < BT / 32; ++wv) t[k] += sm[k][wv];
    double st[kNStat];
    for (int s = 0; s < kNStat; ++s) st[s] = 0.0;
    cons_finish<MODE>(st, i, t[0], t[1], t[2], a.y, a.b, a.sigma, a.z, a.lam);
    for (int s = 0; s < kNStat; ++s) part_long[(int64_t)slot * kNStat + s] = st[s];
  }
  finish_partials(a.fin);
}

// one group per chunk of <= kChunk entries.  Chunks of a long constraint leave their three sums in ch_out
// (k_long_finish adds them in order and finishes the constraint); chunks of C's sym-upper list (line search only)
// go straight into the block's partial row: <C,RR^T>, <C,RD^T> (the entry sum is <C,RD^T+DR^T>, halved) and <C,DD^T>.
template <typename T, int VEC, int GS, int NIT, int MODE>
__global__ void __launch_bounds__(kBlock) k_cons_chunk(const ConsArgs<T> a) {
  ALORA_GRID_DEP();
  constexpr int GPB = kBlock / GS;
  constexpr int NST = 12;
  const int lane = threadIdx.x % GS, grp = threadIdx.x / GS;
  const unsigned gmask = group_mask<GS>();
  double st[NST];
#pragma unroll
  for (int s = 0; s < NST; ++s) st[s] = 0.0;
  for (int64_t c = (int64_t)blockIdx.x * GPB + grp; c < a.nchunk; c += (int64_t)gridDim.x * GPB) {
    const int64_t e0 = __ldg(a.ch_beg + c), e1 = __ldg(a.ch_end + c);
    T s0 = T(0), s1 = T(0), s2 = T(0);
#pragma unroll 4
    for (int64_t e = e0; e < e1; ++e) cons_entry<T, VEC, GS, NIT, MODE>(a, e, lane, s0, s1, s2);
    const double z = group_sum<GS>((double)s0, gmask);
    double q1 = 0.0, q2 = 0.0;
    if (MODE == CONS_LS) { q1 = group_sum<GS>((double)s1, gmask); q2 = group_sum<GS>((double)s2, gmask); }
    if (lane == 0) {
      if (c < a.nchunk_A) { a.ch_out[3 * c] = z; a.ch_out[3 * c + 1] = q1; a.ch_out[3 * c + 2] = q2; }
      else { st[LS_CRR] += z; st[LS_CRD] += 0.5 * q1; st[LS_CDD] += q2; }
    }
  }
  block_reduce_store<NST>(st, a.part_chunk + (int64_t)blockIdx.x * kNStat);
  finish_partials(a.fin);
}

// shapes (GS, NIT) by number of VEC-packs per row
struct Shape { int gs, nit; };
__host__ inline int shape_index(int nvec) {
  if (nvec <= 1) return 0; if (nvec <= 2) return 1; if (nvec <= 4) return 2; if (nvec <= 8) return 3;
  if (nvec <= 16) return 4; if (nvec <= 32) return 5; if (nvec <= 64) return 6; return -1;
}
constexpr Shape kShapes[7] = {{1, 1}, {2, 1}, {4, 1}, {8, 1}, {8, 2}, {16, 2}, {16, 4}};   // k_rows, k_cons
// tiled row kernel: few lanes per row -- the per-row bookkeeping (addresses, scalars, fp64 sums) is issued once
// per group, so fewer lanes per row means fewer warp instructions per row; a lane holds up to 4 packs
constexpr Shape kTShapes[7] = {{1, 1}, {2, 1}, {2, 2}, {4, 2}, {8, 2}, {8, 4}, {16, 4}};     // f + grad, adjoint
// wide ELL (all modes) and the warm line search: more lanes per row (two operands per row or 8 slots per row in registers)
constexpr Shape kTShapesW[7] = {{1, 1}, {2, 1}, {4, 1}, {4, 2}, {8, 2}, {8, 4}, {16, 4}};
// cold line search: as above, but 2 lanes x 2 packs for 3 - 4 packs per row (config 1, r = 16: 46.8 -> 43.1 us once the
// dense variant's bank swizzle made that shape conflict-free; the warm form and the wide variants are slower with it)
constexpr Shape kTShapesLS[7] = {{1, 1}, {2, 1}, {2, 2}, {4, 2}, {8, 2}, {8, 4}, {16, 4}};
__host__ inline Shape tiled_shape(int mode, int idx, bool wide) {
  return (wide || mode == ROWS_LS_WARM) ? kTShapesW[idx] : mode == ROWS_LS_FUSED ? kTShapesLS[idx] : kTShapes[idx];
}

}  // namespace alora
