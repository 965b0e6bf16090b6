// Pass kernels for transform length 160 = 10 x 16, 16 thread(s) per pencil, f32 (see sizes.def).
#define PF_S 160
#define PF_RA 10
#define PF_RB 16
#define PF_TPP 16
#define PF_ONLY_F32
#include "inst.cuh"
