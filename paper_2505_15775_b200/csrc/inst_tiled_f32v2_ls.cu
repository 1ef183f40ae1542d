// tiled row kernel, float rows, 2-element vector loads, line search (cold, warm)
#define ALORA_T float
#define ALORA_VEC 2
#define ALORA_SUF f32v2
#define ALORA_TILED_LS 1
#include "inst_tiled.inc"
