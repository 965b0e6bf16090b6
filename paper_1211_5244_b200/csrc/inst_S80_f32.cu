// Pass kernels for transform length 80 = 20 x 4, 4 thread(s) per pencil, f32 (see sizes.def).
#define PF_S 80
#define PF_RA 20
#define PF_RB 4
#define PF_TPP 4
#define PF_ONLY_F32
#include "inst.cuh"
