// Pass kernels for transform length 120 = 10 x 12, 12 thread(s) per pencil, f64 (see sizes.def).
#define PF_S 120
#define PF_RA 10
#define PF_RB 12
#define PF_TPP 12
#define PF_ONLY_F64
#include "inst.cuh"
