// instantiations of the hot-path kernels for float rows loaded 2 element(s) at a time
#define ALORA_T float
#define ALORA_VEC 2
#define ALORA_SUF f32v2
#include "inst.inc"
