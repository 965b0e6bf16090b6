// Pass kernels for transform length 8 = 8 x 1, 1 thread(s) per pencil, f64 (see sizes.def).
#define PF_S 8
#define PF_RA 8
#define PF_RB 1
#define PF_TPP 1
#define PF_ONLY_F64
#include "inst.cuh"
