// Pass kernels for transform length 400 = 20 x 20, 20 thread(s) per pencil, f64 (see sizes.def).
#define PF_S 400
#define PF_RA 20
#define PF_RB 20
#define PF_TPP 20
#define PF_ONLY_F64
#include "inst.cuh"
