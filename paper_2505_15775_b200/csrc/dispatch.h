// dispatch.h -- host-side launchers for the templated kernels, one translation unit per
// (element type, vector width) so the instantiations compile in parallel.
#pragma once
#include "kernels.cuh"

namespace alora {

#define ALORA_DECL_INST(T, SUF)                                                                       \
  cudaError_t launch_rows_##SUF(int shape, int mode, const RowArgs<T>& a, int grid, cudaStream_t s);  \
  cudaError_t launch_cons1_##SUF(int mode, int single, const ConsArgs<T>& a, int grid, cudaStream_t s); \
  cudaError_t launch_ent_cw_##SUF(int mode, int single, const ConsArgs<T>& a, int grid, cudaStream_t s); \
  cudaError_t launch_cons_##SUF(int shape, int mode, int chunked, const ConsArgs<T>& a, int grid,     \
                                cudaStream_t s);                                                      \
  cudaError_t launch_tiled_##SUF(int shape, int mode, int full, int flags, const RowArgs<T>& a, int grid, cudaStream_t s, int dev); \
  int occ_tiled_##SUF(int shape, int mode, int full, int flags, int64_t ld);                                                      \
  int occ_rows_##SUF(int shape, int mode);                                                            \
  cudaError_t launch_rows_ep_##SUF(int shape, const RowArgs<T>& a, int grid, cudaStream_t s);         \
  cudaError_t launch_rows_cw_##SUF(const RowArgs<T>& a, int grid, cudaStream_t s);                    \
  int occ_rows_cw_##SUF(int nvec);                                                                    \
  int occ_rows_ep_##SUF(int shape);                                                                   \
  cudaError_t launch_rows_seg_##SUF(int shape, const RowArgs<T>& a, int grid, cudaStream_t s);        \
  int occ_cons_##SUF(int shape, int mode, int chunked);

ALORA_DECL_INST(float, f32v4)
ALORA_DECL_INST(float, f32v2)
ALORA_DECL_INST(float, f32v1)
ALORA_DECL_INST(double, f64v2)
ALORA_DECL_INST(double, f64v1)
#undef ALORA_DECL_INST

// generic front-ends: vec = elements per vector load
inline cudaError_t launch_rows(int vec, int shape, int mode, const RowArgs<float>& a, int grid, cudaStream_t s) {
  return vec == 4 ? launch_rows_f32v4(shape, mode, a, grid, s)
       : vec == 2 ? launch_rows_f32v2(shape, mode, a, grid, s) : launch_rows_f32v1(shape, mode, a, grid, s);
}
inline cudaError_t launch_rows(int vec, int shape, int mode, const RowArgs<double>& a, int grid, cudaStream_t s) {
  return vec == 2 ? launch_rows_f64v2(shape, mode, a, grid, s) : launch_rows_f64v1(shape, mode, a, grid, s);
}
inline cudaError_t launch_rows_ep(int vec, int shape, const RowArgs<float>& a, int grid, cudaStream_t s) {
  return vec == 4 ? launch_rows_ep_f32v4(shape, a, grid, s)
       : vec == 2 ? launch_rows_ep_f32v2(shape, a, grid, s) : launch_rows_ep_f32v1(shape, a, grid, s);
}
inline cudaError_t launch_rows_ep(int vec, int shape, const RowArgs<double>& a, int grid, cudaStream_t s) {
  return vec == 2 ? launch_rows_ep_f64v2(shape, a, grid, s) : launch_rows_ep_f64v1(shape, a, grid, s);
}
inline cudaError_t launch_rows_cw(int vec, const RowArgs<float>& a, int grid, cudaStream_t s) {
  return vec == 4 ? launch_rows_cw_f32v4(a, grid, s) : vec == 2 ? launch_rows_cw_f32v2(a, grid, s) : launch_rows_cw_f32v1(a, grid, s);
}
inline cudaError_t launch_rows_cw(int vec, const RowArgs<double>& a, int grid, cudaStream_t s) {
  return vec == 2 ? launch_rows_cw_f64v2(a, grid, s) : launch_rows_cw_f64v1(a, grid, s);
}
inline int occ_rows_cw(float, int vec, int nvec) { return vec == 4 ? occ_rows_cw_f32v4(nvec) : vec == 2 ? occ_rows_cw_f32v2(nvec) : occ_rows_cw_f32v1(nvec); }
inline int occ_rows_cw(double, int vec, int nvec) { return vec == 2 ? occ_rows_cw_f64v2(nvec) : occ_rows_cw_f64v1(nvec); }
inline cudaError_t launch_rows_seg(int vec, int shape, const RowArgs<float>& a, int grid, cudaStream_t s) {
  return vec == 4 ? launch_rows_seg_f32v4(shape, a, grid, s)
       : vec == 2 ? launch_rows_seg_f32v2(shape, a, grid, s) : launch_rows_seg_f32v1(shape, a, grid, s);
}
inline cudaError_t launch_rows_seg(int vec, int shape, const RowArgs<double>& a, int grid, cudaStream_t s) {
  return vec == 2 ? launch_rows_seg_f64v2(shape, a, grid, s) : launch_rows_seg_f64v1(shape, a, grid, s);
}
inline int occ_rows_ep(float, int vec, int shape) {
  return vec == 4 ? occ_rows_ep_f32v4(shape) : vec == 2 ? occ_rows_ep_f32v2(shape) : occ_rows_ep_f32v1(shape);
}
inline int occ_rows_ep(double, int vec, int shape) { return vec == 2 ? occ_rows_ep_f64v2(shape) : occ_rows_ep_f64v1(shape); }
inline cudaError_t launch_ent_cw(int vec, int mode, int single, const ConsArgs<float>& a, int grid, cudaStream_t s) {
  return vec == 4 ? launch_ent_cw_f32v4(mode, single, a, grid, s)
       : vec == 2 ? launch_ent_cw_f32v2(mode, single, a, grid, s) : launch_ent_cw_f32v1(mode, single, a, grid, s);
}
inline cudaError_t launch_ent_cw(int vec, int mode, int single, const ConsArgs<double>& a, int grid, cudaStream_t s) {
  return vec == 2 ? launch_ent_cw_f64v2(mode, single, a, grid, s) : launch_ent_cw_f64v1(mode, single, a, grid, s);
}
inline cudaError_t launch_cons1(int vec, int mode, int single, const ConsArgs<float>& a, int grid, cudaStream_t s) {
  return vec == 4 ? launch_cons1_f32v4(mode, single, a, grid, s)
       : vec == 2 ? launch_cons1_f32v2(mode, single, a, grid, s) : launch_cons1_f32v1(mode, single, a, grid, s);
}
inline cudaError_t launch_cons1(int vec, int mode, int single, const ConsArgs<double>& a, int grid, cudaStream_t s) {
  return vec == 2 ? launch_cons1_f64v2(mode, single, a, grid, s) : launch_cons1_f64v1(mode, single, a, grid, s);
}
inline cudaError_t launch_cons(int vec, int shape, int mode, int chunked, const ConsArgs<float>& a, int grid, cudaStream_t s) {
  return vec == 4 ? launch_cons_f32v4(shape, mode, chunked, a, grid, s)
       : vec == 2 ? launch_cons_f32v2(shape, mode, chunked, a, grid, s) : launch_cons_f32v1(shape, mode, chunked, a, grid, s);
}
inline cudaError_t launch_cons(int vec, int shape, int mode, int chunked, const ConsArgs<double>& a, int grid, cudaStream_t s) {
  return vec == 2 ? launch_cons_f64v2(shape, mode, chunked, a, grid, s) : launch_cons_f64v1(shape, mode, chunked, a, grid, s);
}
inline cudaError_t launch_tiled(int vec, int shape, int mode, int full, int flags, const RowArgs<float>& a, int grid, cudaStream_t s, int dev) {
  return vec == 4 ? launch_tiled_f32v4(shape, mode, full, flags, a, grid, s, dev)
       : vec == 2 ? launch_tiled_f32v2(shape, mode, full, flags, a, grid, s, dev) : launch_tiled_f32v1(shape, mode, full, flags, a, grid, s, dev);
}
inline cudaError_t launch_tiled(int vec, int shape, int mode, int full, int flags, const RowArgs<double>& a, int grid, cudaStream_t s, int dev) {
  return vec == 2 ? launch_tiled_f64v2(shape, mode, full, flags, a, grid, s, dev) : launch_tiled_f64v1(shape, mode, full, flags, a, grid, s, dev);
}
inline int occ_tiled(float, int vec, int shape, int mode, int full, int flags, int64_t ld) {
  return vec == 4 ? occ_tiled_f32v4(shape, mode, full, flags, ld) : vec == 2 ? occ_tiled_f32v2(shape, mode, full, flags, ld) : occ_tiled_f32v1(shape, mode, full, flags, ld);
}
inline int occ_tiled(double, int vec, int shape, int mode, int full, int flags, int64_t ld) {
  return vec == 2 ? occ_tiled_f64v2(shape, mode, full, flags, ld) : occ_tiled_f64v1(shape, mode, full, flags, ld);
}
inline int occ_rows(float, int vec, int shape, int mode) {
  return vec == 4 ? occ_rows_f32v4(shape, mode) : vec == 2 ? occ_rows_f32v2(shape, mode) : occ_rows_f32v1(shape, mode);
}
inline int occ_rows(double, int vec, int shape, int mode) {
  return vec == 2 ? occ_rows_f64v2(shape, mode) : occ_rows_f64v1(shape, mode);
}
inline int occ_cons(float, int vec, int shape, int mode, int ch) {
  return vec == 4 ? occ_cons_f32v4(shape, mode, ch) : vec == 2 ? occ_cons_f32v2(shape, mode, ch) : occ_cons_f32v1(shape, mode, ch);
}
inline int occ_cons(double, int vec, int shape, int mode, int ch) {
  return vec == 2 ? occ_cons_f64v2(shape, mode, ch) : occ_cons_f64v1(shape, mode, ch);
}

}  // namespace alora
