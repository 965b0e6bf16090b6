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

#if defined(__CUDA_ARCH__)
PF_HD void cta_sync() { __syncthreads(); }
#else
void host_cta_sync();  // provided by the development-only host harness
PF_HD void cta_sync() { host_cta_sync(); }
#endif

// ------------------------------------------------------------------ geometry
template <typename T_, int S_, int RA_, int RB_, int TPP_, int P_, bool LANES_P_>
struct Geo {
    using T = T_;
    static constexpr int S = S_, RA = RA_, RB = RB_, TPP = TPP_, P = P_;
    static constexpr bool LANES_P = LANES_P_;
    static_assert(RA * RB == S, "S = RA * RB");
    static_assert(RA % TPP == 0 && RB % TPP == 0, "TPP must divide both radices");
    static constexpr int CA = RB / TPP;  // n1 columns per thread (layout A)
    static constexpr int CB = RA / TPP;  // k2 columns per thread (layout B)
    static constexpr int V = S / TPP;    // complex values per thread
    static constexpr int NT = TPP * P;   // threads per CTA
    static constexpr int RBP = (RB % 2 == 0 && RB > 1) ? RB + 1 : RB;  // odd pitch: conflict-free both ways
    static constexpr int XPITCH = RA * RBP;
    static constexpr int XELEMS = LANES_P ? S * P : P * XPITCH;        // one exchange buffer
    static constexpr size_t SMEM_BYTES = 2 * (size_t)XELEMS * sizeof(cx<T_>);

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
};

// ------------------------------------------------------------------ twiddles kept in registers
template <class G>
struct Twiddles {
    using T = typename G::T;
    static constexpr int NA = G::CA * (G::RA - 1), NB = G::CB * (G::RB - 1);
    cx<T> a[NA > 0 ? NA : 1];  // w^{n1 k2}, n1 = t + TPP i, k2 = 1..RA-1   (forward pass 1)
    cx<T> b[NB > 0 ? NB : 1];  // w^{n1 k2}, k2 = t + TPP i', n1 = 1..RB-1  (inverse pass 1, conjugated on use)
    template <bool NEED_A, bool NEED_B>
    PF_HD void load(const cx<T> *tab, int t) {
        if constexpr (NEED_A && G::RB > 1)
            static_for<G::CA>([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                static_for<G::RA - 1>([&](auto kc) {
                    constexpr int k2 = decltype(kc)::value + 1;
                    a[i * (G::RA - 1) + k2 - 1] = tab[((t + G::TPP * i) * k2) % G::S];
                });
            });
        if constexpr (NEED_B && G::RB > 1)
            static_for<G::CB>([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                static_for<G::RB - 1>([&](auto nc) {
                    constexpr int n1 = decltype(nc)::value + 1;
                    b[i * (G::RB - 1) + n1 - 1] = tab[((t + G::TPP * i) * n1) % G::S];
                });
            });
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
            static_for<RA - 1>([&](auto kc) {
                constexpr int k2 = decltype(kc)::value + 1;
                xb[G::xidx(p, n1, k2)] = u[k2] * tw.a[i * (RA - 1) + k2 - 1];
            });
        }
    });
    if constexpr (RB > 1) {
        cta_sync();
        static_for<G::CB>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            const int k2 = t + G::TPP * i;
            cx<T> *g = v + i * RB;
            static_for<RB>([&](auto nc) { constexpr int n1 = decltype(nc)::value; g[n1] = xb[G::xidx(p, n1, k2)]; });
            dft<T, RB, false>(g);
        });
    }
}

// Inverse, layout B -> layout A.  v[i'*RB + k1] in, v[i*RA + n2] out (n2 < RA/2 only when PRUNED).
template <class G, bool PRUNED>
PF_HD void inv_BtoA(cx<typename G::T> *v, const Twiddles<G> &tw, cx<typename G::T> *xb, int t, int p) {
    using T = typename G::T;
    constexpr int RA = G::RA, RB = G::RB;
    if constexpr (RB > 1) {
        static_for<G::CB>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            const int k2 = t + G::TPP * i;
            cx<T> *g = v + i * RB;
            dft<T, RB, true>(g);
            xb[G::xidx(p, 0, k2)] = g[0];
            static_for<RB - 1>([&](auto nc) {
                constexpr int n1 = decltype(nc)::value + 1;
                xb[G::xidx(p, n1, k2)] = mul_conj(g[n1], tw.b[i * (RB - 1) + n1 - 1]);
            });
        });
        cta_sync();
    }
    static_for<G::CA>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        cx<T> *u = v + i * RA;
        if constexpr (RB > 1) {
            const int n1 = t + G::TPP * i;
            static_for<RA>([&](auto kc) { constexpr int k2 = decltype(kc)::value; u[k2] = xb[G::xidx(p, n1, k2)]; });
        }
        if constexpr (PRUNED) dft_pruned_out<T, RA, true>(u); else dft<T, RA, true>(u);
    });
}

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
template <class G, bool PRUNED>
PF_HD void store_A(const cx<typename G::T> *v, cx<typename G::T> *dst, long long ns, int t, bool valid) {
    constexpr int NA2 = PRUNED ? G::RA / 2 : G::RA;
    if (!valid) return;
    static_for<G::CA>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        static_for<NA2>([&](auto nc) {
            constexpr int n2 = decltype(nc)::value;
            const int n = (t + G::TPP * i) + G::RB * n2;
            dst[n * ns] = v[i * G::RA + n2];
        });
    });
}
// layout B element (i', k1) <-> k = (t + TPP i') + RA k1
template <class G>
PF_HD void load_B(cx<typename G::T> *v, const cx<typename G::T> *src, long long ns, int t, bool valid) {
    using T = typename G::T;
    static_for<G::CB>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        static_for<G::RB>([&](auto kc) {
            constexpr int k1 = decltype(kc)::value;
            const int k = (t + G::TPP * i) + G::RA * k1;
            v[i * G::RB + k1] = valid ? src[k * ns] : mk<T>((T)0, (T)0);
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
            dst[k * ns] = v[i * G::RB + k1];
        });
    });
}

// ------------------------------------------------------------------ pass bodies
// F2: (transpose +) spread + 1D FFT along axis b
template <class G, bool PRUNED>
PF_HD void body_f2(const PassParams &prm, int bid, int nb, int tid, void *smem) {
    using T = typename G::T;
    int t, p; G::split(tid, t, p);
    cx<T> *xb = reinterpret_cast<cx<T> *>(smem);
    Twiddles<G> tw; tw.template load<true, false>(reinterpret_cast<const cx<T> *>(prm.tw), t);
    int par = 0;
    for (int tile = bid; tile < prm.n_tiles; tile += nb, par ^= 1) {
        const int g = tile / prm.tiles_per_g, pp = (tile % prm.tiles_per_g) * G::P + p;
        const bool valid = pp < prm.n_p;
        cx<T> v[G::V];
        load_A<G, PRUNED>(v, reinterpret_cast<const cx<T> *>(prm.in) + g * prm.gs_in + pp * prm.ps_in, prm.ns_in, t, valid);
        fwd_AtoB<G, PRUNED>(v, tw, xb + par * G::XELEMS, t, p);
        store_B<G>(v, reinterpret_cast<cx<T> *>(prm.out) + g * prm.gs_out + pp * prm.ps_out, prm.ns_out, t, valid);
    }
}

// I2: inverse 1D FFT along axis b + compactification (+ transpose)
template <class G, bool PRUNED>
PF_HD void body_i2(const PassParams &prm, int bid, int nb, int tid, void *smem) {
    using T = typename G::T;
    int t, p; G::split(tid, t, p);
    cx<T> *xb = reinterpret_cast<cx<T> *>(smem);
    Twiddles<G> tw; tw.template load<false, true>(reinterpret_cast<const cx<T> *>(prm.tw), t);
    int par = 0;
    for (int tile = bid; tile < prm.n_tiles; tile += nb, par ^= 1) {
        const int g = tile / prm.tiles_per_g, pp = (tile % prm.tiles_per_g) * G::P + p;
        const bool valid = pp < prm.n_p;
        cx<T> v[G::V];
        load_B<G>(v, reinterpret_cast<const cx<T> *>(prm.in) + g * prm.gs_in + pp * prm.ps_in, prm.ns_in, t, valid);
        inv_BtoA<G, PRUNED>(v, tw, xb + par * G::XELEMS, t, p);
        store_A<G, PRUNED>(v, reinterpret_cast<cx<T> *>(prm.out) + g * prm.gs_out + pp * prm.ps_out, prm.ns_out, t, valid);
    }
}

// F3: spread + 1D FFT along axis c, K^F multiply (Eq. 3), inverse 1D FFT along c,
// compactification; in place over the tile it read.
template <class G, bool PRUNED>
PF_HD void body_f3(const PassParams &prm, int bid, int nb, int tid, void *smem) {
    using T = typename G::T;
    int t, p; G::split(tid, t, p);
    cx<T> *xb0 = reinterpret_cast<cx<T> *>(smem), *xb1 = xb0 + G::XELEMS;
    Twiddles<G> tw; tw.template load<true, true>(reinterpret_cast<const cx<T> *>(prm.tw), t);
    const T *kint = reinterpret_cast<const T *>(prm.kint);
    for (int tile = bid; tile < prm.n_tiles; tile += nb) {
        const int g = tile / prm.tiles_per_g, pp = (tile % prm.tiles_per_g) * G::P + p;
        const bool valid = pp < prm.n_p;
        cx<T> v[G::V];
        load_A<G, PRUNED>(v, reinterpret_cast<const cx<T> *>(prm.in) + g * prm.gs_in + pp * prm.ps_in, prm.ns_in, t, valid);
        T kv[G::V];
        const T *kp = kint + (size_t)tile * G::V * G::NT + tid;
        static_for<G::V>([&](auto rc) { constexpr int r = decltype(rc)::value; kv[r] = kp[(size_t)r * G::NT]; });
        fwd_AtoB<G, PRUNED>(v, tw, xb0, t, p);
        static_for<G::V>([&](auto rc) { constexpr int r = decltype(rc)::value; v[r] = scale(v[r], kv[r]); });
        inv_BtoA<G, PRUNED>(v, tw, xb1, t, p);
        store_A<G, PRUNED>(v, reinterpret_cast<cx<T> *>(prm.out) + g * prm.gs_out + pp * prm.ps_out, prm.ns_out, t, valid);
    }
}

// F1: spread + 1D FFT (R2C) along axis a
// Two real pencils adjacent along x are transformed as ONE complex pencil z = rho(2q) + i rho(2q+1)
// (the real array read as complex IS that packing) and separated with the Hermitian symmetry
// F_{S-k} = conj(F_k) of PAPER.md:55; only k = 0..S/2 is kept.  in: pairs, out: complex.
template <class G, bool PRUNED>
PF_HD void body_f1(const PassParams &prm, int bid, int nb, int tid, void *smem) {
    using T = typename G::T;
    static_assert(G::LANES_P, "the R2C pass runs on a strided axis");
    int t, p; G::split(tid, t, p);
    cx<T> *xb0 = reinterpret_cast<cx<T> *>(smem), *xb1 = xb0 + G::XELEMS;
    Twiddles<G> tw; tw.template load<true, false>(reinterpret_cast<const cx<T> *>(prm.tw), t);
    constexpr int S = G::S, NK = S / 2 + 1, NM = (NK + G::TPP - 1) / G::TPP;
    for (int tile = bid; tile < prm.n_tiles; tile += nb) {
        const int g = tile / prm.tiles_per_g, pp = (tile % prm.tiles_per_g) * G::P + p;
        const bool valid = pp < prm.n_p;
        cx<T> v[G::V];
        load_A<G, PRUNED>(v, reinterpret_cast<const cx<T> *>(prm.in) + g * prm.gs_in + pp * prm.ps_in, prm.ns_in, t, valid);
        fwd_AtoB<G, PRUNED>(v, tw, xb0, t, p);
        static_for<G::CB>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            static_for<G::RB>([&](auto kc) {
                constexpr int k1 = decltype(kc)::value;
                xb1[G::nidx(p, (t + G::TPP * i) + G::RA * k1)] = v[i * G::RB + k1];
            });
        });
        cta_sync();
        cx<T> *dst = reinterpret_cast<cx<T> *>(prm.out) + g * prm.gs_out + 2 * pp * prm.ps_out;
        static_for<NM>([&](auto mc) {
            constexpr int m = decltype(mc)::value;
            const int k = t + G::TPP * m;
            if (k < NK && valid) {
                const cx<T> zk = xb1[G::nidx(p, k)], zp = xb1[G::nidx(p, (S - k) % S)];
                const T hf = (T)0.5;
                // A = (Z_k + conj Z_{S-k})/2 ; B = -i (Z_k - conj Z_{S-k})/2
                dst[k * prm.ns_out] = mk<T>(hf * (zk.re + zp.re), hf * (zk.im - zp.im));
                dst[k * prm.ns_out + prm.ps_out] = mk<T>(hf * (zk.im + zp.im), hf * (zp.re - zk.re));
            }
        });
    }
}

// I1: inverse 1D FFT (C2R) along axis a + compactification
// Z_k = A_k + i B_k rebuilt from the half spectra of the two packed pencils (Z_{S-k} = conj A_k + i conj B_k),
// one complex inverse transform, real part -> pencil 2q, imaginary part -> pencil 2q+1.
template <class G, bool PRUNED>
PF_HD void body_i1(const PassParams &prm, int bid, int nb, int tid, void *smem) {
    using T = typename G::T;
    static_assert(G::LANES_P, "the C2R pass runs on a strided axis");
    int t, p; G::split(tid, t, p);
    cx<T> *xb = reinterpret_cast<cx<T> *>(smem);
    Twiddles<G> tw; tw.template load<false, true>(reinterpret_cast<const cx<T> *>(prm.tw), t);
    constexpr int S = G::S;
    int par = 0;
    for (int tile = bid; tile < prm.n_tiles; tile += nb, par ^= 1) {
        const int g = tile / prm.tiles_per_g, pp = (tile % prm.tiles_per_g) * G::P + p;
        const bool valid = pp < prm.n_p;
        cx<T> v[G::V];
        const cx<T> *src = reinterpret_cast<const cx<T> *>(prm.in) + g * prm.gs_in + 2 * pp * prm.ps_in;
        static_for<G::CB>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            static_for<G::RB>([&](auto kc) {
                constexpr int k1 = decltype(kc)::value;
                const int k = (t + G::TPP * i) + G::RA * k1;
                const bool lower = k <= S / 2;
                const int kk = lower ? k : S - k;
                cx<T> a = mk<T>((T)0, (T)0), b = a;
                if (valid) { a = src[kk * prm.ns_in]; b = src[kk * prm.ns_in + prm.ps_in]; }
                v[i * G::RB + k1] = lower ? mk<T>(a.re - b.im, a.im + b.re) : mk<T>(a.re + b.im, b.re - a.im);
            });
        });
        inv_BtoA<G, PRUNED>(v, tw, xb + par * G::XELEMS, t, p);
        store_A<G, PRUNED>(v, reinterpret_cast<cx<T> *>(prm.out) + g * prm.gs_out + pp * prm.ps_out, prm.ns_out, t, valid);
    }
}

}  // namespace pfft
