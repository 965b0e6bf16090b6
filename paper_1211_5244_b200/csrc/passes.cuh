// passes.cuh -- the five fused passes of the customised 3D FFT Poisson solve,
// written once as templates over the transform geometry.
//
// One CTA works on a tile of P pencils of length S = RA * RB.  A pencil is handled by TPP threads;
// every thread keeps V = S / TPP complex values in registers and the only on-chip exchange per 1D
// transform is ONE trip through shared memory between the two register passes:
//
//   layout A (inputs of a forward transform):  thread t holds x[n],  n = n1 + RB*n2,  n1 = t + TPP*i
//   pass 1: DFT_RA over n2 in registers  (pruned when the axis is zero padded -- the paper's "spread")
//           twiddle w_S^{n1*k2}
//   exchange through shared memory
//   pass 2: DFT_RB over n1 in registers
//   layout B (outputs):                        thread t holds X[k],  k = k2 + RA*k1,  k2 = t + TPP*i'
//
// The inverse runs B -> A with conjugated factors and, on a zero-padded axis, only forms the
// outputs n < S/2 (the paper's "compactification").  Global memory is touched straight from /
// into registers: tile rows are whole 128-byte lines, zeros are never read or written.
//
// Two thread mappings share all of the code:
//   LANES_P = true  : consecutive lanes = consecutive pencils (pencils strided in memory, the
//                     pencil index is the contiguous array axis) -- the "transpose" of PAPER.md:53
//                     is nothing but this addressing;
//   LANES_P = false : consecutive lanes = consecutive points of one pencil (transform along the
//                     contiguous array axis).
#pragma once

#include "fft_core.cuh"

namespace pfft {

PF_HD void cta_sync() { __syncthreads(); }
PF_HD void warp_sync() { __syncwarp(); }

enum PassKind { KIND_F1 = 0, KIND_F2 = 1, KIND_F3 = 2, KIND_I2 = 3, KIND_I1 = 4,
                // sharded single solve: F1 / I2 whose stores go straight into the A1 slabs of the peer GPUs
                KIND_F1S = 5, KIND_I2S = 6 };
PF_CE int base_kind(int kind) { return kind == KIND_F1S ? KIND_F1 : (kind == KIND_I2S ? KIND_I2 : kind); }

// Which transforms take two-level inter-pass twiddles (Geo::TW2F / TW2I): fp64, twiddled radix 8 .. 24.  Measured on B200 (DESIGN.md
// section 10c): the load/store pipe is the busiest unit of these kernels (74 % in F3 at S = 256) and 25 % of its work is twiddle loads;
// rows 1, 2, 3, 4, 8, 12 of the table and one more complex multiply per element instead of 15 rows: 128^3 -> 256^3 94.4 -> 90.0 us per
// solve, 256^3 -> 512^3 797 -> 770; radix 24 (8 rows instead of 23): 96^3 -> 192^3 49.2 -> 47.2.  Radix 32 (10 loads, 21 more multiplies)
// loses, fp32 is issue bound: both keep one load per element.
#ifndef PF_TW2
#define PF_TW2 1     // 0: every twiddle from the table (A/B builds)
#endif
#ifndef PF_TW2_MAXR
#define PF_TW2_MAXR 24
#endif
PF_CE bool tw2_radix(int R, int real_bytes) { return PF_TW2 != 0 && real_bytes == 8 && R >= 8 && R <= PF_TW2_MAXR; }

// ------------------------------------------------------------------ geometry
// NBUF_   : exchange buffers (2 = one barrier per exchange, 1 = half the shared memory, one more barrier)
// TWS_    : twiddles w_S^{n1 k2} read from a shared-memory table (true) or held in registers (false)
// MINB_   : __launch_bounds__ minimum resident CTAs per SM (register cap); 0 = automatic
// STG_    : 3 = register double buffer (the next tile is loaded into a second register set while the current one is
//           transformed; no shared memory).  Else asynchronous staging (cp.async, no register cost): 0 = none, tiles are loaded straight into
//           registers; 1 = the NEXT tile's inputs land in a shared-memory stage while the current tile is
//           transformed; 2 = as 1, and pass F3 also stages its K^F values.  Where that stage does not fit next to
//           the exchange buffer (the inverse passes I2 / I1 read S resp. S/2+1 rows), the EXCHANGE BUFFER ITSELF is
//           the stage: it is idle from a tile's last exchange read to the next tile's first exchange write, so the
//           next tile's copies are issued there and land while the last register pass and the stores run
// KLATE_  : pass F3 loads its K^F values right before the multiply (fewer live registers) instead of
//           at the top of the tile
template <typename T_, int S_, int RA_, int RB_, int TPP_, int P_, bool LANES_P_, int NBUF_ = 2, bool TWS_ = true,
          int MINB_ = 0, int STG_ = 0, bool KLATE_ = false>
struct Geo {
    using T = T_;
    static constexpr int S = S_, RA = RA_, RB = RB_, TPP = TPP_, P = P_;
    static constexpr bool LANES_P = LANES_P_;
    static constexpr int NBUF = NBUF_, STG = STG_;
    static constexpr bool KLATE = KLATE_;
    // lanes along the transform: the TPP threads of a pencil sit in one warp, so the exchange is
    // warp-private and a warp-level barrier is enough
    static constexpr bool WARP_LOCAL = !LANES_P_ && (32 % TPP_ == 0);
    static PF_HD void xsync() { if (WARP_LOCAL) warp_sync(); else cta_sync(); }
    static constexpr bool TWS = TWS_ && RB_ > 1;
    // two-level twiddles (shared-memory tables only): w^{n1 k2} = w^{n1 (k2 mod 4)} * w^{n1 4 floor(k2 / 4)} -- rows 1, 2, 3 and
    // 4, 8, 12, ... of the table instead of all of them: 3 + (R - 1) / 4 loads per column instead of R - 1, one more complex
    // multiply for the elements with both factors (tw2_radix)
    static constexpr bool TW2F = TWS && tw2_radix(RA_, (int)sizeof(T_));   // forward direction: the RA outputs of the first pass are twiddled
    static constexpr bool TW2I = TWS && tw2_radix(RB_, (int)sizeof(T_));   // inverse direction: the RB outputs of its first pass
    static_assert(NBUF == 1 || NBUF == 2, "one or two exchange buffers");
    static_assert(RA * RB == S, "S = RA * RB");
    // TPP divides RB; it need not divide RA: a thread then owns ceil(RA / TPP) columns k2 = t + TPP*i of layout B,
    // the last of which exists only for t + TPP*i < RA (b_on).  That is what makes lengths such as 160 = 16 x 10,
    // 320 = 20 x 16 or 768 = 24 x 32 fit two register passes with <= 32 values per thread.
    static_assert(RB % TPP == 0, "TPP must divide the second radix");
    static constexpr int CA = RB / TPP;                  // n1 columns per thread (layout A)
    static constexpr int CB = (RA + TPP - 1) / TPP;      // k2 columns per thread (layout B)
    static constexpr bool RAGGED_B = RA % TPP != 0;
    static constexpr int V = CB * RB;                    // complex values per thread (>= CA * RA = S / TPP)
    template <int I> static PF_HD bool b_on(int t) { return !RAGGED_B || I < CB - 1 || t + TPP_ * I < RA_; }
    static constexpr int NT = TPP * P;   // threads per CTA
    // MINB_ = 0: aim at 512 resident threads per SM (a 128-register budget per thread)
    static constexpr int MINB = MINB_ > 0 ? MINB_ : (512 / NT > 0 ? 512 / NT : 1);
    static constexpr int RBP = (RB % 2 == 0 && RB > 1) ? RB + 1 : RB;  // odd pitch: conflict-free both ways
    static constexpr int XPITCH = RA * RBP;
    static constexpr int XELEMS = LANES_P ? S * P + (STG_ > 0 ? 2 * P : 0) : P * XPITCH;   // one exchange buffer (+ I1's Nyquist row when it doubles as the stage)
    static constexpr int TW_TABLES = !TWS ? 0 : (RA == RB ? 1 : 2);            // [k2][n1] and [n1][k2]
    static constexpr int TW_ELEMS = TW_TABLES * S;
    static constexpr size_t SMEM_BYTES = ((size_t)NBUF * XELEMS + TW_ELEMS) * sizeof(cx<T_>);
    // a one-pass kernel only keeps the table(s) its direction reads: F1/F2 [k2][n1], I2/I1 [n1][k2], F3 both
    static PF_CE int tw_elems(int kind) { return (kind == KIND_F3 ? TW_TABLES : (TW_TABLES > 0 ? 1 : 0)) * S; }
    static PF_CE size_t smem_bytes(int kind) { return ((size_t)NBUF * XELEMS + tw_elems(kind)) * sizeof(cx<T_>); }

    static PF_HD void split(int tid, int &t, int &p) {
        if (LANES_P) { p = tid % P; t = tid / P; } else { t = tid % TPP; p = tid / TPP; }
    }
    // exchange slot of element (n1, k2) of pencil p
    static PF_HD int xidx(int p, int n1, int k2) {
        return LANES_P ? (n1 + RB * k2) * P + p : p * XPITCH + k2 * RBP + n1;
    }
    // natural-order slot k of pencil p (Hermitian split of pass F1)
    static PF_HD int nidx(int p, int k) { return LANES_P ? k * P + p : p * XPITCH + k; }
};

#define PF_MAX_WIDE 32
// Per-launch parameters.  Strides are in elements of the accessed type.
struct PassParams {
    const void *in;
    void *out;
    const void *kint;  // F3 only: internal K^F, [tile][V][NT] reals, pre-scaled
    const void *tw;    // S complex: exp(-2 pi i m / S)
    long long gs_in, ns_in, ps_in;
    long long gs_out, ns_out, ps_out;
    int n_p;           // pencils per g
    int tiles_per_g;   // ceil(n_p / P)
    int n_tiles;       // n_g * tiles_per_g
    int late_tw;       // 1: build the twiddle tables after the first tile's loads have been issued (else before: the PDL order)
    int pdl_trigger;   // programmatic dependent launch: 0 = the next pass may launch from the start of this one, 1 = once this CTA is
                       // past its last tile's loads, 2 = only when this pass exits (the implicit trigger)
    int k_g0;          // F3 of a plane chunk: first plane of the chunk (K^F is indexed by the plane's position in the whole grid)
    int k_fold;        // F3, K^F even along axis b (poisson_set_kernel_even): S_b, the pencils pp > S_b / 2 read the K^F of pencil
                       // S_b - pp and only pencils 0 .. S_b / 2 are stored (k_tpg tiles per plane); 0: every pencil is stored
    int k_tpg;
    int prefetch;      // bit 0: prefetch the next tile's inputs into L2 (unstaged tile loops); bit 1: F3 prefetches its K^F lines
    // several densities per launch (small grids, poisson_solve_batch): tile = bi * n_tiles1 + tile of density bi
    int n_tiles1;      // tiles of ONE density (n_tiles = nb * n_tiles1; nb = 1 for a single solve)
    int use_list;      // 0: in/out + bi * bs_in/bs_out; 1: inputs are blist[bi] (F1: rho); 2: outputs are blist[bi] (I1: V)
    long long bs_in, bs_out;   // elements between the intermediates of consecutive densities
    const void *blist[PF_MAX_WIDE];   // sharded stores (sh_R > 1): base of every rank's destination slab instead
    // sharded single solve: the output array is distributed over sh_R GPUs along a "varying" axis v (F1S: axis a, the planes
    // k_a; I2S: the split axis o of rho / V, sh_total = T points in all), rank s owning a contiguous range of it; the other
    // non-x axis u is whole on every rank.  Destination of element (v, u, x): blist[s] + vl * st_v + u * st_u + x with the
    // strides of a dense [.][.][N_x] array (sh_vslow: v is the slower of the two axes in memory)
    int sh_R, sh_total, sh_vslow, sh_nx, sh_eu;
    int sh_lo[PF_MAX_WIDE + 1];   // rank s owns v in [sh_lo[s], sh_lo[s + 1]) = [floor(T s / R), floor(T (s + 1) / R))
    int sh_u0;         // global u coordinate of this rank's first g (F1S: first o of its slab; I2S: first k_a plane it owns)
    int sh_vp;         // I2S: 1 = the split coordinate v is the pencil index pp and x the transform index n, 0 = the reverse
    // any-length kernel only (generic_pass.cuh): transform length, pencils per tile, radices (product = gen_S), zero-padded axis,
    // real pencils along x of the R2C / C2R pass, complex K^F
    int gen_S, gen_P, gen_nfac, gen_pruned, gen_nreal, gen_kcplx, gen_lanes_p;
    int gen_L, gen_blue;           // buffer / transform length (gen_S, or Bluestein's convolution length M) and the Bluestein flag
    const void *chirp, *bspec;     // Bluestein: exp(-i pi n^2 / S), n < S;  FFT_M of the wrapped conjugate chirp, / M
    int gen_fac[16];
};

template <typename T> PF_HD const cx<T> *pass_in(const PassParams &prm, int bi) {
    return prm.use_list == 1 ? reinterpret_cast<const cx<T> *>(prm.blist[bi]) : reinterpret_cast<const cx<T> *>(prm.in) + bi * prm.bs_in;
}
template <typename T> PF_HD cx<T> *pass_out(const PassParams &prm, int bi) {
    return prm.use_list == 2 ? reinterpret_cast<cx<T> *>(const_cast<void *>(prm.blist[bi])) : reinterpret_cast<cx<T> *>(prm.out) + bi * prm.bs_out;
}

// Sharded stores: address of element (v, u, x) of the distributed output (see PassParams::sh_*).
template <typename T> PF_HD cx<T> *shard_ptr(const PassParams &prm, int v, int u, int x) {
    const int s = ((v + 1) * prm.sh_R - 1) / prm.sh_total;                                 // owner of v (planner.hpp: shard_owner)
    const int lo = prm.sh_lo[s], es = prm.sh_lo[s + 1] - lo, vl = v - lo;                  // rank s holds es points of v
    const long long st_v = prm.sh_vslow ? (long long)prm.sh_eu * prm.sh_nx : prm.sh_nx;
    const long long st_u = prm.sh_vslow ? prm.sh_nx : (long long)es * prm.sh_nx;
    return reinterpret_cast<cx<T> *>(const_cast<void *>(prm.blist[s])) + vl * st_v + u * st_u + x;
}

// ------------------------------------------------------------------ programmatic dependent launch
// Every pass is launched with programmatic stream serialisation: its CTAs may become resident while
// the previous pass drains, run their prologue (twiddle tables: constant data), and only then wait
// for the previous pass's memory to be complete and visible.
PF_HD void pdl_launch_dependents() {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}
PF_HD void pdl_wait_prior_grid() {
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

// ------------------------------------------------------------------ inter-pass twiddles w_S^{n1 k2}
// TWS: two shared-memory tables, [k2][n1] for the forward pass (thread owns n1) and [n1][k2] for the
// inverse pass (thread owns k2), so that consecutive lanes read consecutive entries; one table when
// RA == RB (the table is symmetric).  Otherwise: per-thread register copies.
template <class G>
struct Twiddles {
    using T = typename G::T;
    static constexpr int NA = G::TWS ? 1 : (G::CA * (G::RA - 1) > 0 ? G::CA * (G::RA - 1) : 1);
    static constexpr int NB = G::TWS ? 1 : (G::CB * (G::RB - 1) > 0 ? G::CB * (G::RB - 1) : 1);
    cx<T> a[NA], b[NB];
    const cx<T> *ta, *tb;

    // tab: S entries exp(-2 pi i m / S) in global memory; smem_tw: G::TW_ELEMS entries of shared memory
    template <bool NEED_A, bool NEED_B>
    PF_HD void init(const cx<T> *tab, cx<T> *smem_tw, int tid, int t) {
        constexpr bool ONE = G::TW_TABLES == 1;                       // RA == RB: the table is symmetric
        constexpr bool FILL_A = ONE || NEED_A, FILL_B = !ONE && NEED_B;
        ta = smem_tw; tb = smem_tw + (FILL_A && FILL_B ? G::S : 0);
        if constexpr (G::RB > 1) {
            if constexpr (G::TWS) {
                for (int idx = tid; idx < G::S; idx += G::NT) {
                    const cx<T> w = tab[((idx / G::RB) * (idx % G::RB)) % G::S];
                    if constexpr (FILL_A) smem_tw[idx] = w;                                                        // [k2][n1]
                    if constexpr (FILL_B) smem_tw[(FILL_A ? G::S : 0) + (idx % G::RB) * G::RA + idx / G::RB] = w;  // [n1][k2]
                }
                cta_sync();
            } else {
                if constexpr (NEED_A)
                    static_for<G::CA>([&](auto ic) {
                        constexpr int i = decltype(ic)::value;
                        static_for<G::RA - 1>([&](auto kc) {
                            constexpr int k2 = decltype(kc)::value + 1;
                            a[i * (G::RA - 1) + k2 - 1] = tab[((t + G::TPP * i) * k2) % G::S];
                        });
                    });
                if constexpr (NEED_B)
                    static_for<G::CB>([&](auto ic) {
                        constexpr int i = decltype(ic)::value;
                        static_for<G::RB - 1>([&](auto nc) {
                            constexpr int n1 = decltype(nc)::value + 1;
                            b[i * (G::RB - 1) + n1 - 1] = tab[((t + G::TPP * i) * n1) % G::S];
                        });
                    });
            }
        }
    }
    // forward: thread owns n1 = t + TPP*I, needs w^{n1 K2}
    template <int I, int K2> PF_HD cx<T> fwd(int t) const {
        if constexpr (G::TWS) return ta[K2 * G::RB + t + G::TPP * I];
        else return a[I * (G::RA - 1) + K2 - 1];
    }
    // inverse: thread owns k2 = t + TPP*I, needs w^{N1 k2}
    template <int I, int N1> PF_HD cx<T> inv(int t) const {
        if constexpr (G::TWS) return tb[N1 * G::RA + t + G::TPP * I];
        else return b[I * (G::RB - 1) + N1 - 1];
    }
};

// ------------------------------------------------------------------ the 1D transform engine
// Forward, layout A -> layout B.  v[i*RA + n2] in, v[i'*RB + k1] out.  One cta_sync.
template <class G, bool PRUNED>
PF_HD void fwd_AtoB(cx<typename G::T> *v, const Twiddles<G> &tw, cx<typename G::T> *xb, int t, int p) {
    using T = typename G::T;
    constexpr int RA = G::RA, RB = G::RB;
    static_for<G::CA>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        cx<T> *u = v + i * RA;
        if constexpr (PRUNED) dft_pruned_in<T, RA, false>(u); else dft<T, RA, false>(u);
        if constexpr (RB > 1) {
            const int n1 = t + G::TPP * i;
            xb[G::xidx(p, n1, 0)] = u[0];
            if constexpr (G::TW2F) {
                constexpr int NH = (RA - 1) / 4;
                cx<T> wl[3], wh[NH > 0 ? NH : 1];
                static_for<3>([&](auto jc) { constexpr int j = decltype(jc)::value; if constexpr (j + 1 < RA) wl[j] = tw.template fwd<i, j + 1>(t); });
                static_for<NH>([&](auto ac) { constexpr int a = decltype(ac)::value; wh[a] = tw.template fwd<i, 4 * (a + 1)>(t); });
                static_for<RA - 1>([&](auto kc) {
                    constexpr int k2 = decltype(kc)::value + 1;
                    cx<T> val = u[k2];
                    if constexpr (k2 % 4 != 0) val = val * wl[k2 % 4 - 1];
                    if constexpr (k2 / 4 != 0) val = val * wh[k2 / 4 - 1];
                    xb[G::xidx(p, n1, k2)] = val;
                });
            } else {
                static_for<RA - 1>([&](auto kc) {
                    constexpr int k2 = decltype(kc)::value + 1;
                    xb[G::xidx(p, n1, k2)] = u[k2] * tw.template fwd<i, k2>(t);
                });
            }
        }
    });
    if constexpr (RB > 1) {
        G::xsync();
        static_for<G::CB>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            const int k2 = t + G::TPP * i;
            cx<T> *g = v + i * RB;
            if (G::template b_on<i>(t)) {
                static_for<RB>([&](auto nc) { constexpr int n1 = decltype(nc)::value; g[n1] = xb[G::xidx(p, n1, k2)]; });
                dft<T, RB, false>(g);
            } else {
                static_for<RB>([&](auto nc) { constexpr int n1 = decltype(nc)::value; g[n1] = mk<T>((T)0, (T)0); });
            }
        });
    }
}

// Inverse, layout B -> layout A.  v[i'*RB + k1] in, v[i*RA + n2] out (n2 < RA/2 only when PRUNED).
struct NoHook { PF_HD void operator()() const {} };
// after_read(): called once this thread has read its last exchange value (the exchange-buffer stage hooks in here)
template <class G, bool PRUNED, class Hook = NoHook>
PF_HD void inv_BtoA(cx<typename G::T> *v, const Twiddles<G> &tw, cx<typename G::T> *xb, int t, int p, Hook &&after_read = Hook()) {
    using T = typename G::T;
    constexpr int RA = G::RA, RB = G::RB;
    if constexpr (RB > 1) {
        static_for<G::CB>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            const int k2 = t + G::TPP * i;
            cx<T> *g = v + i * RB;
            if (G::template b_on<i>(t)) {
                dft<T, RB, true>(g);
                xb[G::xidx(p, 0, k2)] = g[0];
                if constexpr (G::TW2I) {
                    constexpr int NH = (RB - 1) / 4;
                    cx<T> wl[3], wh[NH > 0 ? NH : 1];
                    static_for<3>([&](auto jc) { constexpr int j = decltype(jc)::value; if constexpr (j + 1 < RB) wl[j] = tw.template inv<i, j + 1>(t); });
                    static_for<NH>([&](auto ac) { constexpr int a = decltype(ac)::value; wh[a] = tw.template inv<i, 4 * (a + 1)>(t); });
                    static_for<RB - 1>([&](auto nc) {
                        constexpr int n1 = decltype(nc)::value + 1;
                        cx<T> val = g[n1];
                        if constexpr (n1 % 4 != 0) val = mul_conj(val, wl[n1 % 4 - 1]);
                        if constexpr (n1 / 4 != 0) val = mul_conj(val, wh[n1 / 4 - 1]);
                        xb[G::xidx(p, n1, k2)] = val;
                    });
                } else {
                    static_for<RB - 1>([&](auto nc) {
                        constexpr int n1 = decltype(nc)::value + 1;
                        xb[G::xidx(p, n1, k2)] = mul_conj(g[n1], tw.template inv<i, n1>(t));
                    });
                }
            }
        });
        G::xsync();
    }
    if constexpr (RB > 1)
        static_for<G::CA>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            cx<T> *u = v + i * RA;
            const int n1 = t + G::TPP * i;
            static_for<RA>([&](auto kc) { constexpr int k2 = decltype(kc)::value; u[k2] = xb[G::xidx(p, n1, k2)]; });
        });
    after_read();
    static_for<G::CA>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        cx<T> *u = v + i * RA;
        if constexpr (PRUNED) dft_pruned_out<T, RA, true>(u); else dft<T, RA, true>(u);
    });
}

// Exchange-buffer bookkeeping.  NBUF = 2: buffers alternate, the barrier inside each transform is
// enough.  NBUF = 1: one more barrier before the buffer is written again.
template <class G>
struct XBufs {
    using T = typename G::T;
    cx<T> *base;
    int which;
    bool dirty;
    PF_HD explicit XBufs(cx<T> *b) : base(b), which(0), dirty(false) {}
    PF_HD cx<T> *next() {
        if constexpr (G::NBUF == 2) { cx<T> *r = base + which * G::XELEMS; which ^= 1; return r; }
        else { if (dirty) G::xsync(); dirty = true; return base; }
    }
};

// ------------------------------------------------------------------ global <-> register adapters
// layout A element (i, n2) <-> n = (t + TPP i) + RB n2 ; only n2 < NA2 is touched (NA2 = RA/2 when pruned)
template <class G, bool PRUNED, typename E>
PF_HD void load_A(cx<typename G::T> *v, const E *src, long long ns, int t, bool valid) {
    using T = typename G::T;
    constexpr int NA2 = PRUNED ? G::RA / 2 : G::RA;
    static_for<G::CA>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        static_for<NA2>([&](auto nc) {
            constexpr int n2 = decltype(nc)::value;
            const int n = (t + G::TPP * i) + G::RB * n2;
            v[i * G::RA + n2] = valid ? src[n * ns] : mk<T>((T)0, (T)0);
        });
    });
}
template <class G, bool PRUNED, bool STREAM = false>
PF_HD void store_A(const cx<typename G::T> *v, cx<typename G::T> *dst, long long ns, int t, bool valid) {
    constexpr int NA2 = PRUNED ? G::RA / 2 : G::RA;
    if (!valid) return;
    static_for<G::CA>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        static_for<NA2>([&](auto nc) {
            constexpr int n2 = decltype(nc)::value;
            const int n = (t + G::TPP * i) + G::RB * n2;
            st_hint<STREAM>(dst + n * ns, v[i * G::RA + n2]);
        });
    });
}
// layout B element (i', k1) <-> k = (t + TPP i') + RA k1
template <class G, bool STREAM = false>
PF_HD void load_B(cx<typename G::T> *v, const cx<typename G::T> *src, long long ns, int t, bool valid) {
    using T = typename G::T;
    static_for<G::CB>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        static_for<G::RB>([&](auto kc) {
            constexpr int k1 = decltype(kc)::value;
            const int k = (t + G::TPP * i) + G::RA * k1;
            v[i * G::RB + k1] = (valid && G::template b_on<i>(t)) ? ld_hint<STREAM>(src + k * ns) : mk<T>((T)0, (T)0);
        });
    });
}
template <class G>
PF_HD void store_B(const cx<typename G::T> *v, cx<typename G::T> *dst, long long ns, int t, bool valid) {
    if (!valid) return;
    static_for<G::CB>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        static_for<G::RB>([&](auto kc) {
            constexpr int k1 = decltype(kc)::value;
            const int k = (t + G::TPP * i) + G::RA * k1;
            if (G::template b_on<i>(t)) dst[k * ns] = v[i * G::RB + k1];
        });
    });
}

// ------------------------------------------------------------------ asynchronous staging (cp.async / LDGSTS)
// With G::STG > 0 a CTA keeps ONE tile of input in flight in shared memory while it transforms the
// previous one: the copies are issued right after the current tile has been pulled into registers and
// have the whole transform + store of that tile to land, at no register cost.

PF_HD unsigned long long evict_first_policy() {
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// one complex element, global -> shared (16 B: L2 only; 8 B: the only size cp.async.cg does not offer)
template <bool STREAM> PF_HD void cp_async_elem(cx<double> *sdst, const cx<double> *gsrc, unsigned long long pol) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(sdst);
    if constexpr (STREAM) asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;" ::"r"(sa), "l"(gsrc), "l"(pol) : "memory");
    else asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gsrc) : "memory");
}
template <bool STREAM> PF_HD void cp_async_elem(cx<float> *sdst, const cx<float> *gsrc, unsigned long long pol) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(sdst);
    if constexpr (STREAM) asm volatile("cp.async.ca.shared.global.L2::cache_hint [%0], [%1], 8, %2;" ::"r"(sa), "l"(gsrc), "l"(pol) : "memory");
    else asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sa), "l"(gsrc) : "memory");
}
// 16 raw bytes (K^F vectors), evict-first
PF_HD void cp_async_vec16(void *sdst, const void *gsrc, unsigned long long pol) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(sdst);
    asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;" ::"r"(sa), "l"(gsrc), "l"(pol) : "memory");
}
PF_HD void cp_async_commit() {
    asm volatile("cp.async.commit_group;" ::: "memory");
}
template <int N> PF_HD void cp_async_wait() {   // at most N of this thread's newest groups still pending
    asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

// K^F values travel in 16-byte vectors: KVEC consecutive registers r of one thread
template <typename T> struct KVec;
template <> struct KVec<double> { static constexpr int N = 2; using V = double2; };
template <> struct KVec<float>  { static constexpr int N = 4; using V = float4; };
PF_HD void kvec_get(const double2 &v, double *o) { o[0] = v.x; o[1] = v.y; }
PF_HD void kvec_get(const float4 &v, float *o) { o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w; }
PF_HD void prefetch_l2(const void *p) {
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}
template <typename VT> PF_HD VT ld_stream_vec(const VT *p) {
    return __ldcs(p);
}

// Shape of the stage of pass KIND: NR points along the transform x W complex columns.
template <class G, bool PRUNED, int KIND>
struct Stage {
    using T = typename G::T;
    static constexpr int NR = KIND == KIND_I1 ? G::S / 2 + 1 : (KIND == KIND_I2 ? G::S : (PRUNED ? G::S / 2 : G::S));
    static constexpr int W = KIND == KIND_I1 ? 2 * G::P : G::P;
    // staging is dropped where it would not leave room for G::MINB resident CTAs (228 KB per SM, 1 KB
    // reserved per CTA): the occupancy the register budget was chosen for wins
    static constexpr size_t SM_SMEM = 233472, CTA_RESERVED = 1024;
    static PF_CE bool fits(size_t stage_bytes) { return (G::smem_bytes(KIND) + stage_bytes + CTA_RESERVED) * G::MINB <= SM_SMEM; }
    static constexpr bool ON = (G::STG == 1 || G::STG == 2) && fits((size_t)NR * W * sizeof(cx<T>));
    static constexpr bool KON = ON && G::STG == 2 && KIND == KIND_F3 && fits(((size_t)NR * W + G::V * G::NT / 2) * sizeof(cx<T>));
    // exchange buffer as the stage (inverse passes, one exchange buffer)
    // (measured at S = 512 fp64: I2 176 -> 160 us; I1 gets SLOWER this way, 108 -> 118 us -- its 256-bit loads straight
    // into registers beat a trip through shared memory -- so XSTG_I1 stays off)
    static constexpr bool XSTG_I1 = false;
    static constexpr bool XON = (G::STG == 1 || G::STG == 2) && !ON && G::NBUF == 1 && G::RB > 1 && (KIND == KIND_I2 || (XSTG_I1 && KIND == KIND_I1 && G::LANES_P));
    static constexpr int IN_ELEMS = ON ? NR * W : 0;
    static constexpr int K_ELEMS = KON ? G::V * G::NT / 2 : 0;   // V*NT reals
    static constexpr size_t BYTES = (size_t)(IN_ELEMS + K_ELEMS) * sizeof(cx<T>);
    // I1: the two pencils of a pair are de-interleaved so that both reads are contiguous across lanes
    static PF_HD int idx(int col, int n) {
        if constexpr (KIND == KIND_I1) return n * W + (col >> 1) + (col & 1) * G::P;
        else return G::LANES_P ? n * W + col : col * NR + n;
    }
    // inside the exchange buffer a contiguous pencil keeps the exchange pitch, so that a warp's copies stay inside
    // the region its own (warp-private) exchange uses
    static PF_HD int xidx(int col, int n) {
        if constexpr (KIND != KIND_I1 && !G::LANES_P) return col * G::XPITCH + n;
        else return idx(col, n);
    }
};
template <class G, bool PRUNED, int KIND>
constexpr size_t pass_smem_bytes() { return G::smem_bytes(KIND) + Stage<G, PRUNED, KIND>::BYTES; }

// L2 prefetch of one tile's inputs (no registers, no shared memory): one request per 128-byte line.
template <class G, class St>
PF_HD void prefetch_tile_l2(const cx<typename G::T> *src, long long ns, long long ps, int ncols, int tid) {
    constexpr int EPL = 128 / (int)sizeof(cx<typename G::T>);
    if constexpr (G::LANES_P) {   // NR rows of W contiguous elements
        constexpr int LPR = (St::W + EPL - 1) / EPL, TOT = St::NR * LPR, IT = (TOT + G::NT - 1) / G::NT;
        static_for<IT>([&](auto jc) {
            constexpr int j = decltype(jc)::value;
            const int c = tid + G::NT * j, row = c / LPR, l = c % LPR;
            if ((TOT % G::NT == 0 || c < TOT) && l * EPL < ncols) prefetch_l2(src + row * ns + l * EPL);
        });
    } else {                      // pencils of NR contiguous elements
        constexpr int LPP = (St::NR + EPL - 1) / EPL, TOT = G::P * LPP, IT = (TOT + G::NT - 1) / G::NT;
        static_for<IT>([&](auto jc) {
            constexpr int j = decltype(jc)::value;
            const int c = tid + G::NT * j, col = c / LPP, l = c % LPP;
            if ((TOT % G::NT == 0 || c < TOT) && col < ncols) prefetch_l2(src + col * ps + l * EPL);
        });
    }
}

// Issue the copies of one tile.  src = element (row 0, column 0) of the tile; ncols = valid columns
// (ragged last tile).  The threads that later share a barrier scope (CTA, or warp when the exchange
// is warp-private) copy exactly the columns that scope reads.
template <class G, class St, bool STREAM, bool XB = false>
PF_HD void stage_issue(cx<typename G::T> *stage, const cx<typename G::T> *src, long long ns, long long ps, int ncols,
                       int tid, unsigned long long pol) {
    auto sidx = [](int col, int n) { if constexpr (XB) return St::xidx(col, n); else return St::idx(col, n); };
    if constexpr (G::LANES_P) {   // rows of W contiguous elements (ps == 1), stride ns
        constexpr int TOT = St::NR * St::W, IT = (TOT + G::NT - 1) / G::NT;
        static_for<IT>([&](auto jc) {
            constexpr int j = decltype(jc)::value;
            const int c = tid + G::NT * j, row = c / St::W, col = c % St::W;
            if ((TOT % G::NT == 0 || c < TOT) && col < ncols) cp_async_elem<STREAM>(stage + sidx(col, row), src + row * ns + col, pol);
        });
    } else {                      // contiguous pencils (ns == 1), stride ps
        constexpr int GT = G::WARP_LOCAL ? 32 : G::NT, GP = GT / G::TPP;
        constexpr int TOT = GP * St::NR, IT = (TOT + GT - 1) / GT;
        const int grp = tid / GT, l = tid % GT;
        static_for<IT>([&](auto jc) {
            constexpr int j = decltype(jc)::value;
            const int c = l + GT * j, pl = c / St::NR, n = c % St::NR, col = grp * GP + pl;
            if ((TOT % GT == 0 || c < TOT) && col < ncols) cp_async_elem<false>(stage + sidx(col, n), src + col * ps + n, pol);
        });
    }
}

// ------------------------------------------------------------------ tiles
// Persistent tile loop.  issue(tile): start the asynchronous copies of a tile (staged mode only);
// after_first(): hook run once, right after the first tile's loads / copies have been issued (the twiddle tables are built
// there, under the latency of those loads); fetch(buf, tile): tile -> registers (from the stage,
// or straight from global memory when not staged); process(buf, tile): transform and store.
// WAITN = copy groups that may still be pending when a tile's inputs are needed.
struct NoPrefetch { PF_HD void operator()(int) const {} };
template <class G, class Buf, bool STAGED, int WAITN, class Issue, class After, class Fetch, class Process, class Pf = NoPrefetch>
PF_HD void tile_loop(int bid, int nb, int n_tiles, bool trig_late, Issue &&issue, After &&after_first, Fetch &&fetch, Process &&process,
                     Pf &&prefetch_next = Pf()) {
    if constexpr (STAGED) {
        int tile = bid;
        if (tile < n_tiles) issue(tile);
        cp_async_commit();
        after_first();
        for (; tile < n_tiles; tile += nb) {
            Buf cur;
            cp_async_wait<WAITN>();
            G::xsync();                       // every copy of the scope has landed
            fetch(cur, tile);
            G::xsync();                       // stage free again
            if (tile + nb < n_tiles) issue(tile + nb);
            else if (trig_late) pdl_launch_dependents();   // last tile of this CTA: its inputs are in registers
            cp_async_commit();
            process(cur, tile);
        }
    } else if constexpr (G::STG == 3) {   // register double buffer: the next tile's loads are in flight while this one is transformed
        int tile = bid;
        Buf cur;
        if (tile < n_tiles) fetch(cur, tile);
        after_first();
        for (; tile < n_tiles; tile += nb) {
            Buf nxt;
            const bool more = tile + nb < n_tiles;
            if (more) fetch(nxt, tile + nb);
            else if (trig_late) pdl_launch_dependents();
            process(cur, tile);
            if (more) cur = nxt;
        }
    } else {
        bool first = true;
        for (int tile = bid; tile < n_tiles; tile += nb) {
            Buf cur;
            fetch(cur, tile);
            if (first) { after_first(); first = false; }           // the first tile's loads are in flight: run the hook under them
            if (tile + nb < n_tiles) prefetch_next(tile + nb);   // unstaged: at least start the next tile DRAM -> L2
            else if (trig_late) pdl_launch_dependents();         // last tile of this CTA: its loads have been issued
            process(cur, tile);
        }
        if (first) after_first();
        if (trig_late && bid >= n_tiles) pdl_launch_dependents();
    }
}

// Exchange buffer as the stage: process(buf, tile, after_read) calls after_read() once the thread has read its last
// exchange value of the tile; a barrier later the buffer is idle and takes the next tile's copies.
template <class G, class Buf, class Issue, class After, class Fetch, class Process>
PF_HD void tile_loop_x(int bid, int nb, int n_tiles, bool trig_late, Issue &&issue, After &&after_first, Fetch &&fetch, Process &&process) {
    int tile = bid;
    if (tile < n_tiles) issue(tile);
    cp_async_commit();
    after_first();
    for (; tile < n_tiles; tile += nb) {
        Buf cur;
        cp_async_wait<0>();
        G::xsync();                       // every copy of the scope has landed
        fetch(cur, tile);
        G::xsync();                       // buffer free: the transform may write it
        if (trig_late && tile + nb >= n_tiles) pdl_launch_dependents();
        process(cur, tile, [&] {
            G::xsync();                   // every thread of the scope is done reading the exchange
            if (tile + nb < n_tiles) issue(tile + nb);
            cp_async_commit();
        });
    }
}

template <class G, bool PRUNED> struct BufA {   // inputs of a forward transform (layout A, data half only)
    static constexpr int NA2 = PRUNED ? G::RA / 2 : G::RA;
    cx<typename G::T> x[G::CA * NA2];
};
template <class G> struct BufB {                // inputs of an inverse transform (layout B)
    cx<typename G::T> x[G::V];
};
template <class G, bool PRUNED, bool WITH_K> struct BufAK {  // F3: inputs (+ the tile's K^F values)
    static constexpr int NA2 = PRUNED ? G::RA / 2 : G::RA;
    cx<typename G::T> x[G::CA * NA2];
    typename G::T k[WITH_K ? G::V : 1];
};

// layout A inputs straight from global memory
template <class G, bool PRUNED, bool STREAM, class B, typename E>
PF_HD void issue_A(B &b, const E *src, long long ns, int t, bool valid) {
    using T = typename G::T;
    constexpr int NA2 = PRUNED ? G::RA / 2 : G::RA;
    static_for<G::CA>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        static_for<NA2>([&](auto nc) {
            constexpr int n2 = decltype(nc)::value;
            const int n = (t + G::TPP * i) + G::RB * n2;
            b.x[i * NA2 + n2] = valid ? ld_hint<STREAM>(src + n * ns) : mk<T>((T)0, (T)0);
        });
    });
}
// layout A inputs from the stage
template <class G, bool PRUNED, class St, class B>
PF_HD void fetch_A(B &b, const cx<typename G::T> *stage, int t, int p, bool valid) {
    using T = typename G::T;
    constexpr int NA2 = PRUNED ? G::RA / 2 : G::RA;
    static_for<G::CA>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        static_for<NA2>([&](auto nc) {
            constexpr int n2 = decltype(nc)::value;
            const int n = (t + G::TPP * i) + G::RB * n2;
            b.x[i * NA2 + n2] = valid ? stage[St::idx(p, n)] : mk<T>((T)0, (T)0);
        });
    });
}
template <class G, bool PRUNED, class B>
PF_HD void unpack_A(cx<typename G::T> *v, const B &b) {
    constexpr int NA2 = PRUNED ? G::RA / 2 : G::RA;
    static_for<G::CA>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        static_for<NA2>([&](auto nc) { constexpr int n2 = decltype(nc)::value; v[i * G::RA + n2] = b.x[i * NA2 + n2]; });
    });
}

// Where thread (t, p) of `tile` finds its K^F vectors: (tile of the internal copy, thread slot in it).  Plain storage: the
// thread's own tile and slot.  Folded storage (PassParams::k_fold): the tile / slot of the mirror pencil S_b - pp.
template <class G>
PF_HD void kf_slot(const PassParams &prm, int tile, int tid, int t, int p, int &ktile, int &ktid) {
    const int tl1 = tile % prm.n_tiles1;                       // tile within one density
    ktile = tl1 + prm.k_g0 * prm.tiles_per_g; ktid = tid;
    if (prm.k_fold) {
        const int g = tl1 / prm.tiles_per_g, pp = (tl1 % prm.tiles_per_g) * G::P + p;
        int ppk = pp <= prm.k_fold / 2 ? pp : prm.k_fold - pp;
        if (ppk < 0) ppk = 0;                                  // pencils past the end of a ragged tile (never used)
        const int pk = ppk % G::P;
        ktile = (g + prm.k_g0) * prm.k_tpg + ppk / G::P;
        ktid = G::LANES_P ? t * G::P + pk : pk * G::TPP + t;
    }
}

#ifndef PF_KPREF
#define PF_KPREF 1   // pass F3 prefetches its K^F lines into L2 at the top of the tile (where PassParams::prefetch bit 1 is set)
#endif
#ifndef PF_TPREF
#define PF_TPREF 1   // L2 prefetch of the next tile's inputs in the unstaged tile loops
#endif
#define PF_TILE_COORDS                                                                   \
    const int bi = tile / prm.n_tiles1, tl = tile - bi * prm.n_tiles1;                   \
    const int g = tl / prm.tiles_per_g, p0 = (tl % prm.tiles_per_g) * G::P, pp = p0 + p; \
    const bool valid = pp < prm.n_p;                                                     \
    (void)p0; (void)valid; (void)bi;

// ---- per-tile work, shared by the one-pass kernels below and the fused solve kernel (solve_kernel.cuh).
// fetch_*: one tile, global memory -> registers.  process_*: transform the tile and store it.
template <class G> struct TileCtx {          // what a tile function needs besides the pass parameters
    int tid, t, p;
    XBufs<G> xbufs;
    Twiddles<G> tw;
    PF_HD TileCtx(int tid_, cx<typename G::T> *xbase) : tid(tid_), xbufs(xbase) { G::split(tid_, t, p); }
};

template <class G, bool PRUNED, bool STREAM, class Buf>
PF_HD void fetch_fwd(Buf &b, const PassParams &prm, int tile, const TileCtx<G> &c) {   // F1 / F2 / F3 inputs (layout A)
    using T = typename G::T;
    const int t = c.t, p = c.p;
    PF_TILE_COORDS
    issue_A<G, PRUNED, STREAM>(b, pass_in<T>(prm, bi) + g * prm.gs_in + pp * prm.ps_in, prm.ns_in, t, valid);
}
template <class G>
PF_HD void fetch_i2(BufB<G> &b, const PassParams &prm, int tile, const TileCtx<G> &c) {
    using T = typename G::T;
    const int t = c.t, p = c.p;
    PF_TILE_COORDS
    load_B<G, true>(b.x, pass_in<T>(prm, bi) + g * prm.gs_in + pp * prm.ps_in, prm.ns_in, t, valid);  // last read of A2
}
// I1 inputs: Z_k = A_k + i B_k rebuilt from the half spectra of the two packed pencils
// (Z_{S-k} = conj A_k + i conj B_k); ld(kk, a, b) fetches element kk of pencils 2*pp and 2*pp + 1.
template <class G, class Ld>
PF_HD void fetch_i1_with(BufB<G> &b, int t, bool valid, Ld &&ld) {
    using T = typename G::T;
    constexpr int S = G::S;
    static_for<G::CB>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        static_for<G::RB>([&](auto kc) {
            constexpr int k1 = decltype(kc)::value;
            const int k = (t + G::TPP * i) + G::RA * k1;
            const bool lower = k <= S / 2;
            const int kk = lower ? k : S - k;
            cx<T> a = mk<T>((T)0, (T)0), bb = a;
            if (valid && G::template b_on<i>(t)) ld(kk, a, bb);
            b.x[i * G::RB + k1] = lower ? mk<T>(a.re - bb.im, a.im + bb.re) : mk<T>(a.re + bb.im, bb.re - a.im);
        });
    });
}
template <class G>
PF_HD void fetch_i1(BufB<G> &b, const PassParams &prm, int tile, const TileCtx<G> &c) {
    using T = typename G::T;
    const int t = c.t, p = c.p;
    PF_TILE_COORDS
    const cx<T> *src = pass_in<T>(prm, bi) + g * prm.gs_in + 2 * pp * prm.ps_in;
    if (prm.ps_in == 1)   // the two pencils of a pair are adjacent: one access (256-bit in fp64)
        fetch_i1_with<G>(b, t, valid, [&](int kk, cx<T> &a, cx<T> &bb) { ld_pair_stream(src + kk * prm.ns_in, a, bb); });
    else
        fetch_i1_with<G>(b, t, valid, [&](int kk, cx<T> &a, cx<T> &bb) {
            a = ld_stream(src + kk * prm.ns_in); bb = ld_stream(src + kk * prm.ns_in + prm.ps_in);
        });
}

// F2: (transpose +) spread + 1D FFT along axis b
template <class G, bool PRUNED>
PF_HD void process_f2(BufA<G, PRUNED> &b, const PassParams &prm, int tile, TileCtx<G> &c) {
    using T = typename G::T;
    const int t = c.t, p = c.p;
    PF_TILE_COORDS
    cx<T> v[G::V];
    unpack_A<G, PRUNED>(v, b);
    fwd_AtoB<G, PRUNED>(v, c.tw, c.xbufs.next(), t, p);
    store_B<G>(v, pass_out<T>(prm, bi) + g * prm.gs_out + pp * prm.ps_out, prm.ns_out, t, valid);
}
// I2: inverse 1D FFT along axis b + compactification (+ transpose)
template <class G, bool PRUNED, bool SHARD = false, class Hook = NoHook>
PF_HD void process_i2(BufB<G> &b, const PassParams &prm, int tile, TileCtx<G> &c, Hook &&after_read = Hook()) {
    using T = typename G::T;
    const int t = c.t, p = c.p;
    PF_TILE_COORDS
    inv_BtoA<G, PRUNED>(b.x, c.tw, c.xbufs.next(), t, p, after_read);
    if constexpr (SHARD) {   // every element goes to the GPU that owns its point of the split axis
        constexpr int NA2 = PRUNED ? G::RA / 2 : G::RA;
        if (valid)
            static_for<G::CA>([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                static_for<NA2>([&](auto nc) {
                    constexpr int n2 = decltype(nc)::value;
                    const int n = (t + G::TPP * i) + G::RB * n2;
                    *shard_ptr<T>(prm, prm.sh_vp ? pp : n, prm.sh_u0 + g, prm.sh_vp ? n : pp) = b.x[i * G::RA + n2];
                });
            });
    } else {
        store_A<G, PRUNED>(b.x, pass_out<T>(prm, bi) + g * prm.gs_out + pp * prm.ps_out, prm.ns_out, t, valid);
    }
}
// F3: spread + 1D FFT along axis c, K^F multiply (Eq. 3), inverse 1D FFT along c,
// compactification; in place over the tile it read.  kmul(v) multiplies the V
// spectrum values of this thread by their K^F entries.
template <class G, bool PRUNED, class Buf, class KMul>
PF_HD void process_f3(Buf &b, const PassParams &prm, int tile, TileCtx<G> &c, KMul &&kmul) {
    using T = typename G::T;
    const int t = c.t, p = c.p;
    PF_TILE_COORDS
    cx<T> v[G::V];
    unpack_A<G, PRUNED>(v, b);
    fwd_AtoB<G, PRUNED>(v, c.tw, c.xbufs.next(), t, p);
    kmul(v);
    inv_BtoA<G, PRUNED>(v, c.tw, c.xbufs.next(), t, p);
    store_A<G, PRUNED>(v, pass_out<T>(prm, bi) + g * prm.gs_out + pp * prm.ps_out, prm.ns_out, t, valid);
}
// K^F of one tile: internal order [tile][V/KVEC][NT][KVEC] (relayout.cuh), 16-byte vectors per thread
template <class G, class VT>
PF_HD void kmul_vectors(cx<typename G::T> *v, const VT *kp /* vector 0 of this thread */) {
    using T = typename G::T;
    using KV = KVec<T>;
    static_assert(G::V % KV::N == 0, "values per thread must fill whole K^F vectors");
    static_for<G::V / KV::N>([&](auto qc) {
        constexpr int q = decltype(qc)::value;
        T kk[KV::N]; kvec_get(kp[(size_t)q * G::NT], kk);
        static_for<KV::N>([&](auto jc) { constexpr int j = decltype(jc)::value; v[q * KV::N + j] = scale(v[q * KV::N + j], kk[j]); });
    });
}
template <class G>
PF_HD void kmul_global(cx<typename G::T> *v, const void *kint, int tile, int tid) {   // streamed straight from global memory
    using T = typename G::T;
    using KV = KVec<T>;
    const typename KV::V *kp = reinterpret_cast<const typename KV::V *>(kint) + (size_t)tile * (G::V / KV::N) * G::NT + tid;   // tile: within one density
    static_for<G::V / KV::N>([&](auto qc) {
        constexpr int q = decltype(qc)::value;
        T kk[KV::N]; kvec_get(ld_stream_vec(kp + (size_t)q * G::NT), kk);
        static_for<KV::N>([&](auto jc) { constexpr int j = decltype(jc)::value; v[q * KV::N + j] = scale(v[q * KV::N + j], kk[j]); });
    });
}
// F1: spread + 1D FFT (R2C) along axis a
// Two real pencils adjacent along x are transformed as ONE complex pencil z = rho(2q) + i rho(2q+1)
// (the real array read as complex IS that packing) and separated with the Hermitian symmetry
// F_{S-k} = conj(F_k) of PAPER.md:55; only k = 0..S/2 is kept.  in: pairs, out: complex.
template <class G, bool PRUNED, bool SHARD = false>
PF_HD void process_f1(BufA<G, PRUNED> &b, const PassParams &prm, int tile, TileCtx<G> &c) {
    static_assert(G::LANES_P, "the R2C pass runs on a strided axis");
    using T = typename G::T;
    constexpr int S = G::S, NK = S / 2 + 1, NM = (NK + G::TPP - 1) / G::TPP;
    const int t = c.t, p = c.p;
    PF_TILE_COORDS
    cx<T> v[G::V];
    unpack_A<G, PRUNED>(v, b);
    fwd_AtoB<G, PRUNED>(v, c.tw, c.xbufs.next(), t, p);
    cx<T> *xn = c.xbufs.next();
    // A thread's layout-B values are Z_k for k = t + TPP m', m' = i + CB k1 -- exactly the k = t + TPP m it writes out below (when TPP
    // divides RA), so Z_k is already in its registers and only Z_{S-k} has to come from another thread: the exchange carries the upper
    // half of the spectrum (k > S/2) only, half the shared-memory stores and half the loads of a full natural-order exchange.
    constexpr bool LEAN = !G::RAGGED_B && (S / 2) % G::TPP == 0;
    constexpr int HM = S / 2 / G::TPP;        // m' >= HM  <=>  k >= S/2
    static_for<G::CB>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        static_for<G::RB>([&](auto kc) {
            constexpr int k1 = decltype(kc)::value;
            if constexpr (!LEAN || i + G::CB * k1 >= HM)
                if (G::template b_on<i>(t)) xn[G::nidx(p, (t + G::TPP * i) + G::RA * k1)] = v[i * G::RB + k1];
        });
    });
    cta_sync();
    cx<T> *dst = pass_out<T>(prm, bi) + g * prm.gs_out + 2 * pp * prm.ps_out;
    const bool pair_store = prm.ps_out == 1;
    static_for<NM>([&](auto mc) {
        constexpr int m = decltype(mc)::value;
        const int k = t + G::TPP * m;
        if (k < NK && valid) {
            cx<T> zk, zp;
            if constexpr (LEAN) {
                zk = v[(m % G::CB) * G::RB + m / G::CB];
                const cx<T> zr = xn[G::nidx(p, (S - k) % S)];                  // in range for every k (slot 0 is never written: not used)
                zp = (k == 0 || 2 * k == S) ? zk : zr;                         // Z_0 and Z_{S/2} pair with themselves
            } else {
                zk = xn[G::nidx(p, k)]; zp = xn[G::nidx(p, (S - k) % S)];
            }
            const T hf = (T)0.5;
            // A = (Z_k + conj Z_{S-k})/2 ; B = -i (Z_k - conj Z_{S-k})/2
            const cx<T> fa = mk<T>(hf * (zk.re + zp.re), hf * (zk.im - zp.im)), fb = mk<T>(hf * (zk.im + zp.im), hf * (zp.re - zk.re));
            if constexpr (SHARD) st_pair(shard_ptr<T>(prm, k, prm.sh_u0 + g, 2 * pp), fa, fb);   // to the GPU that owns plane k
            else if (pair_store) st_pair(dst + k * prm.ns_out, fa, fb);   // adjacent pencils: one access (256-bit in fp64)
            else { dst[k * prm.ns_out] = fa; dst[k * prm.ns_out + prm.ps_out] = fb; }
        }
    });
}
// I1: inverse 1D FFT (C2R) along axis a + compactification
// one complex inverse transform, real part -> pencil 2q, imaginary part -> pencil 2q+1.
template <class G, bool PRUNED, class Hook = NoHook>
PF_HD void process_i1(BufB<G> &b, const PassParams &prm, int tile, TileCtx<G> &c, Hook &&after_read = Hook()) {
    static_assert(G::LANES_P, "the C2R pass runs on a strided axis");
    using T = typename G::T;
    const int t = c.t, p = c.p;
    PF_TILE_COORDS
    inv_BtoA<G, PRUNED>(b.x, c.tw, c.xbufs.next(), t, p, after_read);
    store_A<G, PRUNED, true>(b.x, pass_out<T>(prm, bi) + g * prm.gs_out + pp * prm.ps_out, prm.ns_out, t, valid);
}

// ------------------------------------------------------------------ one pass per launch
#define PF_BODY_PROLOGUE(NEED_A, NEED_B, KIND)                                                        \
    using T = typename G::T;                                                                          \
    using St = Stage<G, PRUNED, KIND>;                                                                \
    cx<T> *smem_c = reinterpret_cast<cx<T> *>(smem);                                                  \
    TileCtx<G> c(tid, smem_c);                                                                        \
    const int t = c.t, p = c.p;                                                                       \
    cx<T> *stage = smem_c + G::NBUF * G::XELEMS + G::tw_elems(KIND);                                       \
    const unsigned long long pol = (St::ON || St::XON) ? evict_first_policy() : 0ull;                              \
    (void)stage; (void)pol; (void)t; (void)p;                                               \
    if (prm.pdl_trigger == 0) pdl_launch_dependents();                                                \
    auto init_tw = [&] { c.tw.template init<NEED_A, NEED_B>(reinterpret_cast<const cx<T> *>(prm.tw), smem_c + G::NBUF * G::XELEMS, tid, c.t); }; \
    if (!prm.late_tw) init_tw();           /* tables first, then wait for the previous pass (the PDL order) */ \
    pdl_wait_prior_grid();                                                                            \
    auto tw_hook = [&] { if (prm.late_tw) init_tw(); };   /* or: under the latency of the first tile's loads */

template <class G, bool PRUNED>
PF_HD void body_f2(const PassParams &prm, int bid, int nb, int tid, void *smem) {
    PF_BODY_PROLOGUE(true, false, KIND_F2)
    using Buf = BufA<G, PRUNED>;
    tile_loop<G, Buf, St::ON, 0>(bid, nb, prm.n_tiles, prm.pdl_trigger == 1,
        [&](int tile) {
            PF_TILE_COORDS
            stage_issue<G, St, true>(stage, pass_in<T>(prm, bi) + g * prm.gs_in + p0 * prm.ps_in, prm.ns_in, prm.ps_in, prm.n_p - p0, tid, pol);
        },
        tw_hook,
        [&](Buf &b, int tile) {
            if constexpr (St::ON) { PF_TILE_COORDS fetch_A<G, PRUNED, St>(b, stage, t, p, valid); }
            else fetch_fwd<G, PRUNED, true>(b, prm, tile, c);
        },
        [&](Buf &b, int tile) {
            if constexpr (St::ON) c.xbufs.dirty = false;   // the loop's barriers already separate the tiles
            process_f2<G, PRUNED>(b, prm, tile, c);
        },
        [&](int tile) {
            PF_TILE_COORDS
            if (PF_TPREF && (prm.prefetch & 1)) prefetch_tile_l2<G, St>(pass_in<T>(prm, bi) + g * prm.gs_in + p0 * prm.ps_in, prm.ns_in, prm.ps_in, prm.n_p - p0, tid);
        });
}

template <class G, bool PRUNED, bool SHARD = false>
PF_HD void body_i2(const PassParams &prm, int bid, int nb, int tid, void *smem) {
    PF_BODY_PROLOGUE(false, true, KIND_I2)
    using Buf = BufB<G>;
    if constexpr (St::XON) {   // the exchange buffer doubles as the stage
        tile_loop_x<G, Buf>(bid, nb, prm.n_tiles, prm.pdl_trigger == 1,
            [&](int tile) {
                PF_TILE_COORDS
                stage_issue<G, St, true, true>(smem_c, pass_in<T>(prm, bi) + g * prm.gs_in + p0 * prm.ps_in, prm.ns_in, prm.ps_in, prm.n_p - p0, tid, pol);  // last read of A2
                if (PF_TPREF && (prm.prefetch & 1) && tile + nb < prm.n_tiles) {   // and the tile after it starts its way DRAM -> L2
                    const int tile2 = tile + nb;
                    const int bi2 = tile2 / prm.n_tiles1, tl2 = tile2 - bi2 * prm.n_tiles1;
                    const int g2 = tl2 / prm.tiles_per_g, q0 = (tl2 % prm.tiles_per_g) * G::P;
                    prefetch_tile_l2<G, St>(pass_in<T>(prm, bi2) + g2 * prm.gs_in + q0 * prm.ps_in, prm.ns_in, prm.ps_in, prm.n_p - q0, tid);
                }
            },
            tw_hook,
            [&](Buf &b, int tile) {
                PF_TILE_COORDS
                static_for<G::CB>([&](auto ic) {
                    constexpr int i = decltype(ic)::value;
                    static_for<G::RB>([&](auto kc) {
                        constexpr int k1 = decltype(kc)::value;
                        const int k = (t + G::TPP * i) + G::RA * k1;
                        b.x[i * G::RB + k1] = (valid && G::template b_on<i>(t)) ? smem_c[St::xidx(p, k)] : mk<T>((T)0, (T)0);
                    });
                });
            },
            [&](Buf &b, int tile, auto &&after_read) {
                c.xbufs.dirty = false;   // the loop's barriers already separate the tiles
                process_i2<G, PRUNED, SHARD>(b, prm, tile, c, after_read);
            });
        return;
    }
    tile_loop<G, Buf, St::ON, 0>(bid, nb, prm.n_tiles, prm.pdl_trigger == 1,
        [&](int tile) {
            PF_TILE_COORDS
            stage_issue<G, St, true>(stage, pass_in<T>(prm, bi) + g * prm.gs_in + p0 * prm.ps_in, prm.ns_in, prm.ps_in, prm.n_p - p0, tid, pol);  // last read of A2
        },
        tw_hook,
        [&](Buf &b, int tile) {
            if constexpr (St::ON) {
                PF_TILE_COORDS
                static_for<G::CB>([&](auto ic) {
                    constexpr int i = decltype(ic)::value;
                    static_for<G::RB>([&](auto kc) {
                        constexpr int k1 = decltype(kc)::value;
                        const int k = (t + G::TPP * i) + G::RA * k1;
                        b.x[i * G::RB + k1] = (valid && G::template b_on<i>(t)) ? stage[St::idx(p, k)] : mk<T>((T)0, (T)0);
                    });
                });
            } else {
                fetch_i2<G>(b, prm, tile, c);
            }
        },
        [&](Buf &b, int tile) {
            if constexpr (St::ON) c.xbufs.dirty = false;
            process_i2<G, PRUNED, SHARD>(b, prm, tile, c);
        },
        [&](int tile) {
            PF_TILE_COORDS
            if (PF_TPREF && (prm.prefetch & 1)) prefetch_tile_l2<G, St>(pass_in<T>(prm, bi) + g * prm.gs_in + p0 * prm.ps_in, prm.ns_in, prm.ps_in, prm.n_p - p0, tid);
        });
}

template <class G, bool PRUNED>
PF_HD void body_f3(const PassParams &prm, int bid, int nb, int tid, void *smem) {
    PF_BODY_PROLOGUE(true, true, KIND_F3)
    using KV = KVec<T>;
    constexpr int NKV = G::V / KV::N;
    constexpr bool K_EARLY = !St::KON && !G::KLATE;
    constexpr bool KPREF = PF_KPREF != 0;
    using Buf = BufAK<G, PRUNED, K_EARLY>;
    const typename KV::V *kint = reinterpret_cast<const typename KV::V *>(prm.kint);
    typename KV::V *kstage = reinterpret_cast<typename KV::V *>(stage + St::IN_ELEMS);
    (void)kstage;
    auto kf_ptr = [&](int tile) -> const typename KV::V * {   // this thread's first K^F vector of `tile`
        int ktile, ktid;
        kf_slot<G>(prm, tile, tid, t, p, ktile, ktid);
        return kint + (size_t)ktile * NKV * G::NT + ktid;
    };
    auto issue_k = [&](int tile) {
        const typename KV::V *kp = kf_ptr(tile);
        static_for<NKV>([&](auto qc) { constexpr int q = decltype(qc)::value; cp_async_vec16(kstage + q * G::NT + tid, kp + (size_t)q * G::NT, pol); });
    };
    tile_loop<G, Buf, St::ON, (St::KON ? 1 : 0)>(bid, nb, prm.n_tiles, prm.pdl_trigger == 1,
        [&](int tile) {
            PF_TILE_COORDS
            stage_issue<G, St, false>(stage, pass_in<T>(prm, bi) + g * prm.gs_in + p0 * prm.ps_in, prm.ns_in, prm.ps_in, prm.n_p - p0, tid, pol);
        },
        [&] {
            if constexpr (St::KON) { if (bid < prm.n_tiles) issue_k(bid); cp_async_commit(); }
            tw_hook();
        },
        [&](Buf &b, int tile) {
            if constexpr (St::ON) { PF_TILE_COORDS fetch_A<G, PRUNED, St>(b, stage, t, p, valid); }
            else fetch_fwd<G, PRUNED, false>(b, prm, tile, c);
            if (G::KLATE && !St::KON && KPREF && (prm.prefetch & 2)) {   // start this tile's K^F on its way DRAM -> L2 now
                const typename KV::V *kp = kf_ptr(tile);
                static_for<NKV>([&](auto qc) { constexpr int q = decltype(qc)::value; prefetch_l2(kp + (size_t)q * G::NT); });
            }
            if constexpr (K_EARLY) {
                const typename KV::V *kp = kf_ptr(tile);
                static_for<NKV>([&](auto qc) { constexpr int q = decltype(qc)::value; kvec_get(ld_stream_vec(kp + (size_t)q * G::NT), b.k + q * KV::N); });
            }
        },
        [&](Buf &b, int tile) {
            if constexpr (St::ON) c.xbufs.dirty = false;
            process_f3<G, PRUNED>(b, prm, tile, c, [&](cx<T> *v) {
                if constexpr (St::KON) {
                    cp_async_wait<1>();      // everything but the next tile's inputs: this tile's K^F (own copies only)
                    kmul_vectors<G>(v, kstage + tid);
                    if (tile + nb < prm.n_tiles) issue_k(tile + nb);
                    cp_async_commit();
                } else if constexpr (G::KLATE) {
                    int ktile, ktid;
                    kf_slot<G>(prm, tile, tid, t, p, ktile, ktid);
                    kmul_global<G>(v, prm.kint, ktile, ktid);
                } else {
                    static_for<G::V>([&](auto rc) { constexpr int r = decltype(rc)::value; v[r] = scale(v[r], b.k[r]); });
                }
            });
        });   // no next-tile prefetch here: measured slower (512^3 fp32 F3 182 -> 196 us), it competes with the K^F prefetch
}

template <class G, bool PRUNED, bool SHARD = false>
PF_HD void body_f1(const PassParams &prm, int bid, int nb, int tid, void *smem) {
    PF_BODY_PROLOGUE(true, false, KIND_F1)
    using Buf = BufA<G, PRUNED>;
    tile_loop<G, Buf, St::ON, 0>(bid, nb, prm.n_tiles, prm.pdl_trigger == 1,
        [&](int tile) {
            PF_TILE_COORDS
            stage_issue<G, St, true>(stage, pass_in<T>(prm, bi) + g * prm.gs_in + p0 * prm.ps_in, prm.ns_in, prm.ps_in, prm.n_p - p0, tid, pol);
        },
        tw_hook,
        [&](Buf &b, int tile) {
            if constexpr (St::ON) { PF_TILE_COORDS fetch_A<G, PRUNED, St>(b, stage, t, p, valid); }
            else fetch_fwd<G, PRUNED, true>(b, prm, tile, c);
        },
        [&](Buf &b, int tile) {
            if constexpr (St::ON) c.xbufs.dirty = false;
            process_f1<G, PRUNED, SHARD>(b, prm, tile, c);
        },
        [&](int tile) {
            PF_TILE_COORDS
            if (PF_TPREF && (prm.prefetch & 1)) prefetch_tile_l2<G, St>(pass_in<T>(prm, bi) + g * prm.gs_in + p0 * prm.ps_in, prm.ns_in, prm.ps_in, prm.n_p - p0, tid);
        });
}

template <class G, bool PRUNED>
PF_HD void body_i1(const PassParams &prm, int bid, int nb, int tid, void *smem) {
    PF_BODY_PROLOGUE(false, true, KIND_I1)
    using Buf = BufB<G>;
    if constexpr (St::XON) {   // the exchange buffer doubles as the stage
        tile_loop_x<G, Buf>(bid, nb, prm.n_tiles, prm.pdl_trigger == 1,
            [&](int tile) {
                PF_TILE_COORDS
                stage_issue<G, St, true, true>(smem_c, pass_in<T>(prm, bi) + g * prm.gs_in + 2 * p0 * prm.ps_in, prm.ns_in, prm.ps_in, 2 * (prm.n_p - p0), tid, pol);
            },
            tw_hook,
            [&](Buf &b, int tile) {
                PF_TILE_COORDS
                fetch_i1_with<G>(b, t, valid, [&](int kk, cx<T> &a, cx<T> &bb) { a = smem_c[St::xidx(2 * p, kk)]; bb = smem_c[St::xidx(2 * p + 1, kk)]; });
            },
            [&](Buf &b, int tile, auto &&after_read) {
                c.xbufs.dirty = false;
                process_i1<G, PRUNED>(b, prm, tile, c, after_read);
            });
        return;
    }
    tile_loop<G, Buf, St::ON, 0>(bid, nb, prm.n_tiles, prm.pdl_trigger == 1,
        [&](int tile) {
            PF_TILE_COORDS   // stage rows: kk = 0..S/2, columns: the 2 P complex pencils of the P pairs
            stage_issue<G, St, true>(stage, pass_in<T>(prm, bi) + g * prm.gs_in + 2 * p0 * prm.ps_in, prm.ns_in, prm.ps_in, 2 * (prm.n_p - p0), tid, pol);
        },
        tw_hook,
        [&](Buf &b, int tile) {
            if constexpr (St::ON) {
                PF_TILE_COORDS
                fetch_i1_with<G>(b, t, valid, [&](int kk, cx<T> &a, cx<T> &bb) { a = stage[St::idx(2 * p, kk)]; bb = stage[St::idx(2 * p + 1, kk)]; });
            } else {
                fetch_i1<G>(b, prm, tile, c);
            }
        },
        [&](Buf &b, int tile) {
            if constexpr (St::ON) c.xbufs.dirty = false;
            process_i1<G, PRUNED>(b, prm, tile, c);
        },
        [&](int tile) {
            PF_TILE_COORDS
            if (PF_TPREF && (prm.prefetch & 1)) prefetch_tile_l2<G, St>(pass_in<T>(prm, bi) + g * prm.gs_in + 2 * p0 * prm.ps_in, prm.ns_in, prm.ps_in, 2 * (prm.n_p - p0), tid);
        });
}

}  // namespace pfft
