// Pass kernels for transform length 36 = 6 x 6, 3 thread(s) per pencil, f64 (see sizes.def).
#define PF_S 36
#define PF_RA 6
#define PF_RB 6
#define PF_TPP 3
#define PF_ONLY_F64
#include "inst.cuh"
