// tiled row kernel, float rows, 2-element vector loads, f + grad and adjoint
#define ALORA_T float
#define ALORA_VEC 2
#define ALORA_SUF f32v2
#define ALORA_TILED_LS 0
#include "inst_tiled.inc"
