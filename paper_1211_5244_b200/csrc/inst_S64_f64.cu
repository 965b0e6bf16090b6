// Pass kernels for transform length 64 = 8 x 8, 8 thread(s) per pencil, f64 (see sizes.def).
#define PF_S 64
#define PF_RA 8
#define PF_RB 8
#define PF_TPP 8
#define PF_ONLY_F64
#include "inst.cuh"
