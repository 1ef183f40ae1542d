// tiled row kernel, double rows, 2-element vector loads, line search (cold, warm)
#define ALORA_T double
#define ALORA_VEC 2
#define ALORA_SUF f64v2
#define ALORA_TILED_LS 1
#include "inst_tiled.inc"
