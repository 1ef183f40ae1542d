// tiled row kernel, float rows, 4-element vector loads, line search (cold, warm)
#define ALORA_T float
#define ALORA_VEC 4
#define ALORA_SUF f32v4
#define ALORA_TILED_LS 1
#include "inst_tiled.inc"
