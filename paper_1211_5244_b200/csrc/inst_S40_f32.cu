// Pass kernels for transform length 40 = 10 x 4, 2 thread(s) per pencil, f32 (see sizes.def).
#define PF_S 40
#define PF_RA 10
#define PF_RB 4
#define PF_TPP 2
#define PF_ONLY_F32
#include "inst.cuh"
