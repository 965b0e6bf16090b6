// Pass kernels for transform length 256 = 16 x 16, 16 thread(s) per pencil, f64 (see sizes.def).
#define PF_S 256
#define PF_RA 16
#define PF_RB 16
#define PF_TPP 16
#define PF_ONLY_F64
#include "inst.cuh"
