// Pass kernels for transform length 96 = 12 x 8, 4 thread(s) per pencil, f32 (see sizes.def).
#define PF_S 96
#define PF_RA 12
#define PF_RB 8
#define PF_TPP 4
#define PF_ONLY_F32
#include "inst.cuh"
