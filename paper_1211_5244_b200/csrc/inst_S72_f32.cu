// Pass kernels for transform length 72 = 12 x 6, 6 thread(s) per pencil, f32 (see sizes.def).
#define PF_S 72
#define PF_RA 12
#define PF_RB 6
#define PF_TPP 6
#define PF_ONLY_F32
#include "inst.cuh"
