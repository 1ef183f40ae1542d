// instantiations of the hot-path kernels for double rows loaded 2 element(s) at a time
#define ALORA_T double
#define ALORA_VEC 2
#define ALORA_SUF f64v2
#include "inst.inc"
