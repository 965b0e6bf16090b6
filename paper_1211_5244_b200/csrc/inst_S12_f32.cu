// Pass kernels for transform length 12 = 12 x 1, 1 thread(s) per pencil, f32 (see sizes.def).
#define PF_S 12
#define PF_RA 12
#define PF_RB 1
#define PF_TPP 1
#define PF_ONLY_F32
#include "inst.cuh"
