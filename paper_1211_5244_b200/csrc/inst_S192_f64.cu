// Pass kernels for transform length 192 = 24 x 8, 8 thread(s) per pencil, f64 (see sizes.def).
#define PF_S 192
#define PF_RA 24
#define PF_RB 8
#define PF_TPP 8
#define PF_ONLY_F64
// 24 complex fp64 values per thread: a 168-register budget (3 CTAs of 128 threads per SM) instead of the default 128
// (measured on the wire configuration: I2 16.5 -> 14.7 us, batched solve 59.2 -> 52.4 us; 12 x 16 with 16 threads per
// pencil is faster in F2 / I2 but slower in F3: 55.5 us)
#define PF_MINB 3
// second factorization 12 x 16 with 16 threads per pencil (variant 9): faster for F2 / I2 (14.4 vs 16.1 / 15.1 us on the wire
// configuration), slower for F3 (32.7 vs 28.8 us); api.cu picks it for those two passes
#define PF_ALT_GEOMETRY pfft::reg_length<double, 192, 12, 16, 16, 1, true, 0, 0, true>(0, 9);
#include "inst.cuh"
