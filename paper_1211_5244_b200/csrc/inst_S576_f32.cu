// Pass kernels for transform length 576 = 24 x 24, 24 thread(s) per pencil, f32 (see sizes.def).
#define PF_S 576
#define PF_RA 24
#define PF_RB 24
#define PF_TPP 24
#define PF_ONLY_F32
#include "inst.cuh"
