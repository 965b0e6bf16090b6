// Pass kernels for transform length 256 = 16 x 16, 16 thread(s) per pencil, f64 (see sizes.def).
#define PF_S 256
#define PF_RA 16
#define PF_RB 16
#define PF_TPP 16
#define PF_ONLY_F64
// tuning experiments: PF_VARIANT(id, NBUF, TWS, MINB, STG, KLATE)
// (instantiated only when the library is built with -DPF_EXPERIMENTS: python -m paper_1211_5244_b200.build --experiments)
#if defined(PF_EXPERIMENTS)
#define PF_EXTRA_VARIANTS PF_VARIANT(1, 2, false, 1, 0, false) PF_VARIANT(2, 1, true, 0, 1, true) PF_VARIANT(3, 1, true, 5, 0, true) \
    PF_VARIANT(4, 1, true, 3, 1, true) PF_VARIANT(5, 1, true, 3, 2, false) PF_VARIANT(6, 1, true, 3, 0, true)
#endif
#include "inst.cuh"
