// Pass kernels for transform length 640 = 20 x 32, 32 thread(s) per pencil, f64 (see sizes.def).
#define PF_S 640
#define PF_RA 20
#define PF_RB 32
#define PF_TPP 32
#define PF_ONLY_F64
// 32 values per thread, 32 threads per pencil: one CTA per SM
#define PF_MINB 1
#define PF_STG 1
#include "inst.cuh"
