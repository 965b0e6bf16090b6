// Pass kernels for transform length 480 = 20 x 24, 24 thread(s) per pencil, f64 (see sizes.def).
#define PF_S 480
#define PF_RA 20
#define PF_RB 24
#define PF_TPP 24
#define PF_ONLY_F64
#include "inst.cuh"
