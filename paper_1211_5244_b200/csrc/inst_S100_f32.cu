// Pass kernels for transform length 100 = 10 x 10, 5 thread(s) per pencil, f32 (see sizes.def).
#define PF_S 100
#define PF_RA 10
#define PF_RB 10
#define PF_TPP 5
#define PF_ONLY_F32
#include "inst.cuh"
