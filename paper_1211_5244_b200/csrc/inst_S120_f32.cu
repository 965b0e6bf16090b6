// Pass kernels for transform length 120 = 12 x 10, 10 thread(s) per pencil, f32 (see sizes.def).
#define PF_S 120
#define PF_RA 12
#define PF_RB 10
#define PF_TPP 10
#define PF_ONLY_F32
#include "inst.cuh"
