// Pass kernels for transform length 60 = 10 x 6, 6 thread(s) per pencil, f32 (see sizes.def).
#define PF_S 60
#define PF_RA 10
#define PF_RB 6
#define PF_TPP 6
#define PF_ONLY_F32
#include "inst.cuh"
