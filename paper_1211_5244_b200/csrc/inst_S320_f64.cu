// Pass kernels for transform length 320 = 16 x 20, 20 thread(s) per pencil, f64 (see sizes.def).
// (RA < RB = TPP: every thread owns one column of the second pass, 16 of 20 threads have one)
#define PF_S 320
#define PF_RA 16
#define PF_RB 20
#define PF_TPP 20
#define PF_ONLY_F64
#include "inst.cuh"
