// tiled row kernel, float rows, 1-element vector loads, line search (cold, warm)
#define ALORA_T float
#define ALORA_VEC 1
#define ALORA_SUF f32v1
#define ALORA_TILED_LS 1
#include "inst_tiled.inc"
