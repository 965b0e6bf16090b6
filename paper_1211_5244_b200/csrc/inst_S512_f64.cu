// Pass kernels for transform length 512 = 32 x 16, 16 thread(s) per pencil, f64 (see sizes.def).
#define PF_S 512
#define PF_RA 32
#define PF_RB 16
#define PF_TPP 16
#define PF_ONLY_F64
// 32 complex fp64 values per thread: needs the full register file, 2 CTAs per SM
#define PF_MINB 2
#include "inst.cuh"
