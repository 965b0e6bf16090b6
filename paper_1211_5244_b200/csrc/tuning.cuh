// tuning.cuh -- per-length tuning knobs of the pass kernels.  build.py generates one translation unit per
// (transform length, precision) from sizes.def:
//     #define PF_S / PF_RA / PF_RB / PF_TPP      (the PF_SIZE line)
//     #define PF_ONLY_F64 | PF_ONLY_F32
//     #include "tuning.cuh"                       (this file: knobs that differ from the defaults of inst.cuh)
//     #include "inst.cuh"
// Knobs (defaults in inst.cuh): PF_NBUF, PF_TWS, PF_MINB, PF_STG, PF_KLATE, PF_PCMUL, PF_ALT_GEOMETRY,
// PF_EXTRA_VARIANTS (tuning experiments, only with -DPF_EXPERIMENTS: python -m paper_1211_5244_b200.build --experiments;
// PF_VARIANT(id, NBUF, TWS, MINB, STG, KLATE) / PF_VARIANT_PC(..., PCMUL), selected with POISSON_VARIANT).
// Every number quoted below was measured on one B200.
#pragma once

#if PF_S == 192 && defined(PF_ONLY_F64)
// 24 complex fp64 values per thread: a 168-register budget (3 CTAs of 128 threads per SM) instead of the default 128
// (measured on the wire configuration: I2 16.5 -> 14.7 us, batched solve 59.2 -> 52.4 us; 12 x 16 with 16 threads per
// pencil is faster in F2 / I2 but slower in F3: 55.5 us)
#define PF_MINB 3
// second factorization 12 x 16 with 16 threads per pencil (variant 9): faster for F2 / I2 (14.4 vs 16.1 / 15.1 us on the wire
// configuration), slower for F3 (32.7 vs 28.8 us); api.cu (preferred_variant) picks it for those two passes
#define PF_ALT_GEOMETRY pfft::reg_length<double, 192, 12, 16, 16, 1, true, 0, 0, true>(0, 9);
#endif

#if PF_S == 256 && defined(PF_ONLY_F64) && defined(PF_EXPERIMENTS)
#define PF_EXTRA_VARIANTS PF_VARIANT(1, 2, false, 1, 0, false) PF_VARIANT(2, 1, true, 0, 1, true) PF_VARIANT(3, 1, true, 5, 0, true) \
    PF_VARIANT(4, 1, true, 3, 1, true) PF_VARIANT(5, 1, true, 3, 2, false) PF_VARIANT(6, 1, true, 3, 0, true) \
    PF_VARIANT(7, 1, true, 0, 3, true) PF_VARIANT(8, 1, true, 3, 3, true) PF_VARIANT(10, 1, false, 3, 0, true) PF_VARIANT(11, 1, false, 4, 0, true)
#endif

#if PF_S == 28 && defined(PF_ONLY_F64)
// one thread per pencil, 28 complex fp64 values in registers (radix 28): no 128-register cap (it spills 256 bytes)
#define PF_MINB 2
#endif

#if PF_S == 448 && defined(PF_ONLY_F64)
// 32 complex fp64 values per thread (28 x 16, two columns of the second pass per thread): as 384 / 512
#define PF_MINB 2
#define PF_STG 1
#endif

#if PF_S == 336 && defined(PF_ONLY_F64)
// 24 complex fp64 values per thread, 192 threads per CTA: as 576
#define PF_MINB 2
#define PF_STG 1
#endif

#if PF_S == 896
// as 1024: one CTA per SM (fp64: 32 complex values per thread, next tile staged)
#define PF_MINB 1
#if defined(PF_ONLY_F64)
#define PF_STG 1
#endif
#endif

#if PF_S == 384 && defined(PF_ONLY_F64)
// 32 complex fp64 values per thread: the full register file, 2 CTAs of 128 threads per SM
#define PF_MINB 2
#define PF_STG 1
#endif

#if PF_S == 512 && defined(PF_ONLY_F64)
// 32 complex fp64 values per thread: needs the full register file, 2 CTAs (8 warps) per SM.  With that few warps
// the global-memory latency is exposed, so the next tile's inputs are staged with cp.async while the current tile is
// transformed (STG = 1; c4a 978 -> 915 us per solve), and the contiguous-axis kernels run as ONE 256-thread CTA per SM
// (PCMUL = 2) so that a single copy of the twiddle tables leaves room for F3's stage.
#define PF_MINB 2
#define PF_STG 1
#define PF_PCMUL 2
#if defined(PF_EXPERIMENTS)
#define PF_EXTRA_VARIANTS PF_VARIANT(1, 1, true, 2, 0, true) PF_VARIANT_PC(3, 1, true, 3, 0, true, 3)
#endif
#endif

#if PF_S == 512 && defined(PF_ONLY_F32) && defined(PF_EXPERIMENTS)
#define PF_EXTRA_VARIANTS PF_VARIANT(1, 1, true, 2, 1, true) PF_VARIANT_PC(2, 1, true, 2, 1, true, 2) PF_VARIANT(3, 1, true, 3, 0, true) \
    PF_VARIANT_PC(4, 1, true, 2, 2, true, 2)
#endif

#if PF_S == 576 && defined(PF_ONLY_F64)
// 24 complex fp64 values per thread: 170 registers, 2 CTAs of 192 threads per SM
#define PF_MINB 2
#define PF_STG 1
#endif

#if (PF_S == 640 || PF_S == 768)
// 32 values per thread, 32 threads per pencil: one CTA per SM (fp64: the next tile staged with cp.async)
#define PF_MINB 1
#if defined(PF_ONLY_F64)
#define PF_STG 1
#endif
#endif

#if PF_S == 1024
// 128 KB exchange buffer: one CTA per SM (fp64: 32 complex values per thread, 256 threads, next tile staged)
#define PF_MINB 1
#if defined(PF_ONLY_F64)
#define PF_STG 1
#endif
#endif
