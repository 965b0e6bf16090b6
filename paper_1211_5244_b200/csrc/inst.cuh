// inst.cuh -- instantiates and registers every pass kernel for ONE transform length.
// An inst_S<len>_<prec>.cu file defines PF_S, PF_RA, PF_RB, PF_TPP (and optionally the tuning knobs
// PF_NBUF, PF_TWS, PF_MINB, PF_STG, PF_KLATE, PF_PCMUL, PF_EXTRA_VARIANTS) and includes this header.
#pragma once

#include "passes.cuh"
#include "registry.hpp"

namespace pfft {

template <class G, bool PRUNED, int KIND>
__global__ void __launch_bounds__(G::NT, G::MINB) pass_kernel(const PassParams prm) {
    extern __shared__ __align__(16) unsigned char pf_smem[];
    const int bid = blockIdx.x, nb = gridDim.x, tid = threadIdx.x;
    if constexpr (KIND == KIND_F1) body_f1<G, PRUNED>(prm, bid, nb, tid, pf_smem);
    else if constexpr (KIND == KIND_F2) body_f2<G, PRUNED>(prm, bid, nb, tid, pf_smem);
    else if constexpr (KIND == KIND_F3) body_f3<G, PRUNED>(prm, bid, nb, tid, pf_smem);
    else if constexpr (KIND == KIND_I2) body_i2<G, PRUNED>(prm, bid, nb, tid, pf_smem);
    else if constexpr (KIND == KIND_F1S) body_f1<G, PRUNED, true>(prm, bid, nb, tid, pf_smem);
    else if constexpr (KIND == KIND_I2S) body_i2<G, PRUNED, true>(prm, bid, nb, tid, pf_smem);
    else body_i1<G, PRUNED>(prm, bid, nb, tid, pf_smem);
}

template <class G, bool PRUNED, int KIND>
static void reg_one(int prec, int variant) {
    KernelEntry e{};
    e.kind = KIND; e.S = G::S; e.pruned = PRUNED ? 1 : 0; e.lanes_p = G::LANES_P ? 1 : 0; e.prec = prec;
    e.variant = variant; e.nbuf = G::NBUF; e.tws = G::TWS ? 1 : 0; e.minb = G::MINB; e.stg = G::STG;
    e.RA = G::RA; e.RB = G::RB;
    e.P = G::P; e.TPP = G::TPP; e.V = G::V; e.NT = G::NT; e.smem_bytes = pass_smem_bytes<G, PRUNED, base_kind(KIND)>();
    e.func = reinterpret_cast<const void *>(&pass_kernel<G, PRUNED, KIND>);
    kernel_registry().push_back(e);
}

// pencils per CTA: whole 128-byte tile rows, >= 128 threads per CTA, whole warps
template <typename T, int TPP>
constexpr int pencils_per_cta() {
    constexpr int by_line = 128 / (int)sizeof(cx<T>);
    int P = by_line;
    while (P * TPP < 128 || (P * TPP) % 32 != 0) P += by_line;
    return P;
}

// PCMUL: the contiguous-axis kernels (lanes along the transform, warp-private exchange) may take PCMUL times
// more pencils per CTA, with MINB / PCMUL resident CTAs: same warps per SM, but ONE copy of the twiddle
// tables per SM, which is what leaves room for the asynchronous stage at S = 512 in fp64.
template <typename T, int S, int RA, int RB, int TPP, int NBUF, bool TWS, int MINB, int STG, bool KLATE, int PCMUL = 1>
static void reg_length(int prec, int variant) {
    constexpr int P = pencils_per_cta<T, TPP>();
    constexpr int MINBC = MINB > 0 ? (MINB / PCMUL > 0 ? MINB / PCMUL : 1) : 0;
    using GP = Geo<T, S, RA, RB, TPP, P, true, NBUF, TWS, MINB, STG, KLATE>;
    using GC = Geo<T, S, RA, RB, TPP, P * PCMUL, false, NBUF, TWS, MINBC, STG, KLATE>;
    reg_one<GP, true, KIND_F1>(prec, variant);  reg_one<GP, false, KIND_F1>(prec, variant);
    reg_one<GP, true, KIND_I1>(prec, variant);  reg_one<GP, false, KIND_I1>(prec, variant);
    reg_one<GP, true, KIND_F2>(prec, variant);  reg_one<GP, false, KIND_F2>(prec, variant);
    reg_one<GP, true, KIND_I2>(prec, variant);  reg_one<GP, false, KIND_I2>(prec, variant);
    reg_one<GP, true, KIND_F3>(prec, variant);  reg_one<GP, false, KIND_F3>(prec, variant);
    reg_one<GC, true, KIND_F2>(prec, variant);  reg_one<GC, false, KIND_F2>(prec, variant);
    reg_one<GC, true, KIND_I2>(prec, variant);  reg_one<GC, false, KIND_I2>(prec, variant);
    reg_one<GC, true, KIND_F3>(prec, variant);  reg_one<GC, false, KIND_F3>(prec, variant);
    if (variant == 0) {   // sharded single solve: F1 / I2 with their stores scattered over the peer GPUs (default geometry only)
        reg_one<GP, true, KIND_F1S>(prec, variant);  reg_one<GP, false, KIND_F1S>(prec, variant);
        reg_one<GP, true, KIND_I2S>(prec, variant);  reg_one<GP, false, KIND_I2S>(prec, variant);
        reg_one<GC, true, KIND_I2S>(prec, variant);  reg_one<GC, false, KIND_I2S>(prec, variant);
    }
}

}  // namespace pfft

#if defined(PF_S)
#ifndef PF_NBUF
#define PF_NBUF 1
#endif
#ifndef PF_TWS
#define PF_TWS true
#endif
#ifndef PF_MINB
#define PF_MINB 0
#endif
#ifndef PF_STG
#define PF_STG 0
#endif
#ifndef PF_KLATE
#define PF_KLATE true
#endif
#ifndef PF_PCMUL
#define PF_PCMUL 1
#endif
#if defined(PF_ONLY_F64)
#define PF_T double
#define PF_PREC 0
#else
#define PF_T float
#define PF_PREC 1
#endif
namespace {
struct PfRegistrar {
    PfRegistrar() {
        pfft::reg_length<PF_T, PF_S, PF_RA, PF_RB, PF_TPP, PF_NBUF, PF_TWS, PF_MINB, PF_STG, PF_KLATE, PF_PCMUL>(PF_PREC, 0);
#if defined(PF_ALT_GEOMETRY)
        PF_ALT_GEOMETRY   // a second factorization of the same length, registered under its own variant id (api.cu: preferred_variant)
#endif
#if defined(PF_EXTRA_VARIANTS)
#define PF_VARIANT(ID, NBUF, TWS, MINB, STG, KLATE) pfft::reg_length<PF_T, PF_S, PF_RA, PF_RB, PF_TPP, NBUF, TWS, MINB, STG, KLATE>(PF_PREC, ID);
#define PF_VARIANT_PC(ID, NBUF, TWS, MINB, STG, KLATE, PCMUL) pfft::reg_length<PF_T, PF_S, PF_RA, PF_RB, PF_TPP, NBUF, TWS, MINB, STG, KLATE, PCMUL>(PF_PREC, ID);
        PF_EXTRA_VARIANTS
#undef PF_VARIANT_PC
#undef PF_VARIANT
#endif
    }
};
static PfRegistrar pf_registrar_instance;
}  // namespace
#endif
