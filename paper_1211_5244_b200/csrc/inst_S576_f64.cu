// Pass kernels for transform length 576 = 24 x 24, 24 thread(s) per pencil, f64 (see sizes.def).
#define PF_S 576
#define PF_RA 24
#define PF_RB 24
#define PF_TPP 24
#define PF_ONLY_F64
// 24 complex fp64 values per thread: 170 registers, 2 CTAs of 192 threads per SM
#define PF_MINB 2
#define PF_STG 1
#include "inst.cuh"
