// Pass kernels for transform length 160 = 16 x 10, 10 thread(s) per pencil, f32 (see sizes.def).
#define PF_S 160
#define PF_RA 16
#define PF_RB 10
#define PF_TPP 10
#define PF_ONLY_F32
#include "inst.cuh"
