// instantiations of the hot-path kernels for float rows loaded 4 element(s) at a time
#define ALORA_T float
#define ALORA_VEC 4
#define ALORA_SUF f32v4
#include "inst.inc"
