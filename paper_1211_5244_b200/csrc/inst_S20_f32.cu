// Pass kernels for transform length 20 = 20 x 1, 1 thread(s) per pencil, f32 (see sizes.def).
#define PF_S 20
#define PF_RA 20
#define PF_RB 1
#define PF_TPP 1
#define PF_ONLY_F32
#include "inst.cuh"
