// tiled row kernel, double rows, 1-element vector loads, line search (cold, warm)
#define ALORA_T double
#define ALORA_VEC 1
#define ALORA_SUF f64v1
#define ALORA_TILED_LS 1
#include "inst_tiled.inc"
