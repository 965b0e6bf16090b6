// Pass kernels for transform length 512 = 32 x 16, 16 thread(s) per pencil, f64 (see sizes.def).
#define PF_S 512
#define PF_RA 32
#define PF_RB 16
#define PF_TPP 16
#define PF_ONLY_F64
// 32 complex fp64 values per thread: needs the full register file, 2 CTAs (8 warps) per SM.  With that few warps
// the global-memory latency is exposed, so the next tile's inputs are staged with cp.async while the current tile is
// transformed (STG = 1; c4a 978 -> 915 us per solve), and the contiguous-axis kernels run as ONE 256-thread CTA per SM
// (PCMUL = 2) so that a single copy of the twiddle tables leaves room for F3's stage.
#define PF_MINB 2
#define PF_STG 1
#define PF_PCMUL 2
// tuning experiments: PF_VARIANT(id, NBUF, TWS, MINB, STG, KLATE) / PF_VARIANT_PC(..., PCMUL)
// (instantiated only when the library is built with -DPF_EXPERIMENTS: python -m paper_1211_5244_b200.build --experiments)
#if defined(PF_EXPERIMENTS)
#define PF_EXTRA_VARIANTS PF_VARIANT(1, 1, true, 2, 0, true) PF_VARIANT_PC(3, 1, true, 3, 0, true, 3)
#endif
#include "inst.cuh"
