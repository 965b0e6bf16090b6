// fused_inst.cuh -- instantiates and registers fused solve kernels (solve_kernel.cuh).
// A fused_*.cu file lists the combinations it holds with PF_FUSED(T, prec, SA, PA, SB, PB, LB, SC, PC, LC, MINB):
//   S* = transform length of axis a / b / c, P* = 1 when that axis is zero padded (pruned transform),
//   LB / LC = 1 when pass F2 / F3 runs on a strided axis (lanes along pencils), 0 on the contiguous axis,
//   MINB = resident CTAs per SM the register budget is cut for.
#pragma once

#include "inst.cuh"
#include "solve_kernel.cuh"

namespace pfft {

template <int S> struct SizeCfg;
#define PF_SIZE(S_, RA_, RB_, TPP_) \
    template <> struct SizeCfg<S_> { static constexpr int RA = RA_, RB = RB_, TPP = TPP_; };
#include "sizes.def"
#undef PF_SIZE

// geometry of one axis inside the fused kernel: one exchange buffer, shared-memory twiddles, no staging, late K^F
template <typename T, int S, bool LANES_P, int MINB>
using FusedGeo = Geo<T, S, SizeCfg<S>::RA, SizeCfg<S>::RB, SizeCfg<S>::TPP, pencils_per_cta<T, SizeCfg<S>::TPP>(), LANES_P,
                     1, true, MINB, 0, true>;

template <typename T, int SA, bool PA, int SB, bool PB, bool LB, int SC, bool PC, bool LC, int MINB>
static void reg_fused(int prec) {
    using GA = FusedGeo<T, SA, true, MINB>;
    using GB = FusedGeo<T, SB, LB, MINB>;
    using GC = FusedGeo<T, SC, LC, MINB>;
    FusedEntry e;
    e.prec = prec;
    e.S[0] = SA; e.S[1] = SB; e.S[2] = SC;
    e.pruned[0] = PA; e.pruned[1] = PB; e.pruned[2] = PC;
    e.lanes_p[0] = 1; e.lanes_p[1] = LB; e.lanes_p[2] = LC;
    e.P[0] = GA::P; e.P[1] = GB::P; e.P[2] = GC::P;
    e.NT = GA::NT; e.minb = GA::MINB;
    e.smem_bytes = SolveSmem<GA, GB, GC>::BYTES;
    e.func = reinterpret_cast<const void *>(&solve_kernel<GA, PA, GB, PB, GC, PC>);
    fused_registry().push_back(e);
}

}  // namespace pfft

#define PF_FUSED(T, PREC, SA, PA, SB, PB, LB, SC, PC, LC, MINB) pfft::reg_fused<T, SA, PA, SB, PB, LB, SC, PC, LC, MINB>(PREC);
namespace {
struct PfFusedRegistrar { PfFusedRegistrar() { PF_FUSED_LIST } };
static PfFusedRegistrar pf_fused_registrar_instance;
}  // namespace
