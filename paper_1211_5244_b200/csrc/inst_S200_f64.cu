// Pass kernels for transform length 200 = 20 x 10, 10 thread(s) per pencil, f64 (see sizes.def).
#define PF_S 200
#define PF_RA 20
#define PF_RB 10
#define PF_TPP 10
#define PF_ONLY_F64
#include "inst.cuh"
