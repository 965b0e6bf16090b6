// Pass kernels for transform length 384 = 24 x 16, 16 thread(s) per pencil, f64 (see sizes.def).
#define PF_S 384
#define PF_RA 24
#define PF_RB 16
#define PF_TPP 16
#define PF_ONLY_F64
// 32 complex fp64 values per thread: the full register file, 2 CTAs of 128 threads per SM
#define PF_MINB 2
#define PF_STG 1
#include "inst.cuh"
