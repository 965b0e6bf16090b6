// Pass kernels for transform length 1024 = 32 x 32, 32 thread(s) per pencil, f64 (see sizes.def).
#define PF_S 1024
#define PF_RA 32
#define PF_RB 32
#define PF_TPP 32
#define PF_ONLY_F64
// 32 complex fp64 values per thread and a 128 KB exchange buffer: one 256-thread CTA per SM
#define PF_MINB 1
#define PF_STG 1
#include "inst.cuh"
