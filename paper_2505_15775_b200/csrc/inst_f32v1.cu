// instantiations of the hot-path kernels for float rows loaded 1 element(s) at a time
#define ALORA_T float
#define ALORA_VEC 1
#define ALORA_SUF f32v1
#include "inst.inc"
