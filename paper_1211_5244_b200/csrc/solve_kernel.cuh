// solve_kernel.cuh -- the whole solve (all 13 steps) as ONE persistent cooperative kernel.
//
//   phase 1   F1 tiles (R2C along axis a)                                  rho -> A1
//   --- grid barrier: every F2 pencil needs every F1 tile (the one all-to-all of a 3D FFT)
//   phase 2   F2 -> F3 -> I2, pipelined per plane g = k_a                  A1 -> A2 -> A2 -> A1
//             F3 of plane g only needs the F2 tiles of plane g, I2 of plane g only the F3 tiles of
//             plane g, so the three passes run as a dataflow: work items are ordered
//                 step s:  F2 tiles of plane s | F3 tiles of plane s-D | I2 tiles of plane s-2D
//             and handed out round-robin to the resident CTAs; an item waits on a per-plane counter
//             (almost never: the skew D covers the items in flight).  A plane of A2 is written,
//             transformed in place and consumed within a few microseconds, i.e. while it is still in
//             the 126 MB L2 -- on grids whose A2 does not fit in L2 (512^3 padded: 539 MB) its four
//             sweeps stop being HBM traffic.
//   --- grid barrier
//   phase 3   I1 tiles (C2R along axis a)                                  A1 -> V
//
// One launch per solve instead of five: no launch gaps, no ramp-up / tail per pass.  The item order is a
// topological order of the dependency graph and every CTA takes its items in increasing order, so with
// all CTAs co-resident (cooperative launch, grid <= resident capacity) the waits cannot deadlock.
#pragma once

#include "passes.cuh"

namespace pfft {

struct SolveParams {
    PassParams pass[5];
    unsigned *sync;   // [0] grid-barrier arrivals, [1] unused, [2 + g] F2 tiles done of plane g, [2 + G + g] F3 tiles done; zero at launch
    int n_planes;     // G = H = S_a/2 + 1
    int t2, t3;       // tiles per plane of F2 / I2 and of F3
    int skew;         // D
};

__device__ __forceinline__ unsigned ld_acquire_gpu(const unsigned *p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
// all threads of the CTA: the CTA's earlier global writes become visible device-wide, then count up
__device__ __forceinline__ void cta_signal(unsigned *ctr) {
    __syncthreads();
    if (threadIdx.x == 0) { __threadfence(); atomicAdd(ctr, 1u); }
}
// all threads of the CTA: block until *ctr >= target, then see everything signalled before
__device__ __forceinline__ void cta_wait(const unsigned *ctr, unsigned target) {
    if (threadIdx.x == 0) {
        // bounded: with all CTAs co-resident and the counters zeroed before the launch the wait is short; if it is not
        // (a bug), fail the launch with a trap -- the host then sees POISSON_ECUDA -- instead of hanging the device
        unsigned spins = 0;
        while (ld_acquire_gpu(ctr) < target) { __nanosleep(40); if (++spins > (1u << 26)) __trap(); }
        __threadfence();
    }
    __syncthreads();
}
__device__ __forceinline__ void grid_barrier(unsigned *ctr, unsigned target) {
    cta_signal(ctr);
    cta_wait(ctr, target);
}

template <class GA, class GB, class GC>
struct SolveSmem {
    using T = typename GA::T;
    static constexpr int maxi(int a, int b) { return a > b ? a : b; }
    static constexpr int X_ELEMS = maxi(GA::NBUF * GA::XELEMS, maxi(GB::NBUF * GB::XELEMS, GC::NBUF * GC::XELEMS));
    // axes with the same factorisation share one twiddle table
    template <class G1, class G2> static constexpr bool same_tables() { return G1::S == G2::S && G1::RA == G2::RA && G1::RB == G2::RB; }
    static constexpr bool B_IS_A = same_tables<GB, GA>(), C_IS_A = same_tables<GC, GA>(), C_IS_B = same_tables<GC, GB>();
    static constexpr int TWA = X_ELEMS;
    static constexpr int TWB = B_IS_A ? TWA : TWA + GA::TW_ELEMS;
    static constexpr int END_B = B_IS_A ? TWA + GA::TW_ELEMS : TWB + GB::TW_ELEMS;
    static constexpr int TWC = C_IS_A ? TWA : (C_IS_B ? TWB : END_B);
    static constexpr int END_C = (C_IS_A || C_IS_B) ? END_B : TWC + GC::TW_ELEMS;
    static constexpr size_t BYTES = (size_t)END_C * sizeof(cx<T>);
};

template <class GA, bool PA, class GB, bool PB, class GC, bool PC>
__global__ void __launch_bounds__(GA::NT, GA::MINB) solve_kernel(const SolveParams prm) {
    static_assert(GA::NT == GB::NT && GA::NT == GC::NT, "the three geometries share one CTA shape");
    static_assert((GA::TWS || GA::RB == 1) && (GB::TWS || GB::RB == 1) && (GC::TWS || GC::RB == 1), "twiddles live in shared memory");
    static_assert(GA::STG == 0 && GB::STG == 0 && GC::STG == 0, "tiles go straight to registers here");
    using T = typename GA::T;
    using SM = SolveSmem<GA, GB, GC>;
    extern __shared__ __align__(16) unsigned char pf_smem[];
    cx<T> *smem_c = reinterpret_cast<cx<T> *>(pf_smem);
    const int bid = blockIdx.x, nb = gridDim.x, tid = threadIdx.x;

    TileCtx<GA> ca(tid, smem_c);
    TileCtx<GB> cb(tid, smem_c);
    TileCtx<GC> cc(tid, smem_c);
    ca.tw.template init<true, true>(reinterpret_cast<const cx<T> *>(prm.pass[KIND_F1].tw), smem_c + SM::TWA, tid, ca.t);
    cb.tw.template init<true, true>(reinterpret_cast<const cx<T> *>(prm.pass[KIND_F2].tw), smem_c + SM::TWB, tid, cb.t);
    cc.tw.template init<true, true>(reinterpret_cast<const cx<T> *>(prm.pass[KIND_F3].tw), smem_c + SM::TWC, tid, cc.t);
    __syncthreads();

    // ---------------- phase 1: F1
    {
        const PassParams &q = prm.pass[KIND_F1];
        for (int tile = bid; tile < q.n_tiles; tile += nb) {
            BufA<GA, PA> b;
            fetch_fwd<GA, PA, true>(b, q, tile, ca);
            process_f1<GA, PA>(b, q, tile, ca);
        }
    }
    grid_barrier(prm.sync, (unsigned)nb);

    // ---------------- phase 2: F2 -> F3 -> I2 per plane
    {
        const int G = prm.n_planes, T2 = prm.t2, T3 = prm.t3, D = prm.skew;
        const int U = 2 * T2 + T3;
        const long long n_items = (long long)(G + 2 * D) * U;
        unsigned *cnt2 = prm.sync + 2, *cnt3 = prm.sync + 2 + G;
        for (long long it = bid; it < n_items; it += nb) {
            const int s = (int)(it / U), r = (int)(it % U);
            if (r < T2) {                                            // F2 of plane s
                const int g = s;
                if (g >= G) continue;
                __syncthreads();                                     // exchange buffer free again
                cb.xbufs.dirty = false;
                const PassParams &q = prm.pass[KIND_F2];
                BufA<GB, PB> b;
                fetch_fwd<GB, PB, true>(b, q, g * T2 + r, cb);
                process_f2<GB, PB>(b, q, g * T2 + r, cb);
                cta_signal(cnt2 + g);
            } else if (r < T2 + T3) {                                // F3 of plane s - D
                const int g = s - D, j = r - T2;
                if (g < 0 || g >= G) continue;
                cta_wait(cnt2 + g, (unsigned)T2);
                cc.xbufs.dirty = false;
                const PassParams &q = prm.pass[KIND_F3];
                const int tile = g * T3 + j;
                BufAK<GC, PC, false> b;
                fetch_fwd<GC, PC, false>(b, q, tile, cc);
                process_f3<GC, PC>(b, q, tile, cc, [&](cx<T> *v) { kmul_global<GC>(v, q.kint, tile, tid); });
                cta_signal(cnt3 + g);
            } else {                                                 // I2 of plane s - 2D
                const int g = s - 2 * D, j = r - T2 - T3;
                if (g < 0 || g >= G) continue;
                cta_wait(cnt3 + g, (unsigned)T3);
                cb.xbufs.dirty = false;
                const PassParams &q = prm.pass[KIND_I2];
                BufB<GB> b;
                fetch_i2<GB>(b, q, g * T2 + j, cb);
                process_i2<GB, PB>(b, q, g * T2 + j, cb);
            }
        }
    }
    grid_barrier(prm.sync, 2u * (unsigned)nb);

    // ---------------- phase 3: I1
    {
        ca.xbufs.dirty = false;
        const PassParams &q = prm.pass[KIND_I1];
        for (int tile = bid; tile < q.n_tiles; tile += nb) {
            BufB<GA> b;
            fetch_i1<GA>(b, q, tile, ca);
            process_i1<GA, PA>(b, q, tile, ca);
        }
    }

    // the counters are zeroed by a cudaMemsetAsync queued before every launch (api.cu: run_fused)
}

}  // namespace pfft
