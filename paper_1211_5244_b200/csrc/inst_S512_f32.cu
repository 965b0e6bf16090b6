// Pass kernels for transform length 512 = 32 x 16, 16 thread(s) per pencil, f32 (see sizes.def).
#define PF_S 512
#define PF_RA 32
#define PF_RB 16
#define PF_TPP 16
#define PF_ONLY_F32
// tuning experiments: PF_VARIANT(id, NBUF, TWS, MINB, STG, KLATE) / PF_VARIANT_PC(..., PCMUL)
// (instantiated only when the library is built with -DPF_EXPERIMENTS: python -m paper_1211_5244_b200.build --experiments)
#if defined(PF_EXPERIMENTS)
#define PF_EXTRA_VARIANTS PF_VARIANT(1, 1, true, 2, 1, true) PF_VARIANT_PC(2, 1, true, 2, 1, true, 2) PF_VARIANT(3, 1, true, 3, 0, true) \
    PF_VARIANT_PC(4, 1, true, 2, 2, true, 2)
#endif
#include "inst.cuh"
