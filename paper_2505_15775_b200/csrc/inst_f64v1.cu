// instantiations of the hot-path kernels for double rows loaded 1 element(s) at a time
#define ALORA_T double
#define ALORA_VEC 1
#define ALORA_SUF f64v1
#include "inst.inc"
