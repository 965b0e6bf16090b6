// generic_pass.cuh -- the five fused passes for ANY transform length ("general sizes":
// PAPER.md:89 "various grid sizes ... maximal for large power of two sizes").
//
// The register engine of passes.cuh is compiled for the lengths of sizes.def (two register passes, S = RA * RB).
// Every other length -- odd N, factors 7, 11, 13, ..., three or more radices (300, 360, 600, 720, 900), primes and
// 2 * prime -- runs here: ONE kernel per (precision, pass kind) whose transform length, tile width and radix list are
// run-time values.  A CTA holds a tile of P pencils x S points in shared memory and runs a Stockham autosort
// mixed-radix FFT on it:
//
//     n = S, s = 1;  for every radix R of S (product of the radices = S):   m = n / R
//         y[q + s (R j + k)] = w_n^{j k}  sum_{r < R}  x[q + s (j + m r)]  w_R^{r k}      j < m, q < s, k < R
//         swap(x, y);  n = m;  s = s R
//
// (natural order in, natural order out, no bit reversal).  The radices are chosen by the plan from {16, 15, 14, 12, 10, 8, 6, 5, 4,
// 3, 2} (the in-register DFTs of fft_core.cuh: a thread holds a whole butterfly), 7 / 11 / 13 (the R-term sums written
// out in registers) and, for any other prime factor p, a fallback that forms one output per thread per step -- O(p) per
// point.  Lengths up to 1024 with a prime factor >= 17 instead take Bluestein's chirp-z (gen_transform below): two smooth
// transforms of length M >= 2S - 1, so that every length is O(S log S).  Twiddles come from the plan's
// table exp(-2 pi i m / S) in shared memory.  The paper's spread / compactification are the zero fill of
// the tile's upper half on load and the store of the lower half only; R2C / C2R pack two real pencils
// adjacent in x into one complex transform exactly as passes.cuh does, with an unpaired last pencil when N_x is odd.
// The same kernel multiplies by a COMPLEX K^F (poisson_set_kernel_complex: kernels without K(-r) = K(r)).
#pragma once

#include "passes.cuh"

namespace pfft {

constexpr int GEN_NT = 256;          // threads per CTA
constexpr int GEN_MAX_S = 4096;      // longest generic transform (three S-point arrays per pencil must fit shared memory)

// tile pitch: odd number of elements, so that both "lanes along pencils" and "lanes along the transform" spread over banks
PF_CE int gen_pitch(int P) { return (P % 2 == 0) ? P + 1 : P; }
PF_CE size_t gen_smem_bytes(int L, int P, size_t cplx_bytes) { return ((size_t)2 * L * gen_pitch(P) + L) * cplx_bytes; }   // L: buffer length (S, or Bluestein's M)

// floor(n / d) for the index ranges of a tile (n d < 2^32) without an integer division: n * ceil(2^32 / d) >> 32
struct GenDiv {
    unsigned d, magic;
    PF_HD explicit GenDiv(int d_) : d((unsigned)d_), magic(d_ > 1 ? 0xFFFFFFFFu / (unsigned)d_ + 1u : 0u) {}
    PF_HD int div(int n) const { return d > 1 ? (int)__umulhi((unsigned)n, magic) : n; }
};

template <typename T> PF_HD cx<T> gen_w(const cx<T> *tw, int i, bool inv) { const cx<T> w = tw[i]; return inv ? conj(w) : w; }

// Radix-R butterfly for a prime R without a literal-twiddle DFT in fft_core.cuh (7, 11, 13): the R-term sums written out
// with the factors w_R^{rk} = w_S^{(S/R)(rk mod R)} read from the shared-memory table.
template <typename T, int R, bool INV>
PF_HD void gen_dft_prime(cx<T> *a, const cx<T> *tw, int wr) {
    cx<T> o[R];
    static_for<R>([&](auto kc) {
        constexpr int k = decltype(kc)::value;
        cx<T> acc = a[0];
        static_for<R - 1>([&](auto rc) {
            constexpr int r = decltype(rc)::value + 1;
            const cx<T> w = gen_w(tw, wr * ((r * k) % R), INV);
            acc = k == 0 ? acc + a[r] : acc + a[r] * w;
        });
        o[k] = acc;
    });
    static_for<R>([&](auto kc) { constexpr int k = decltype(kc)::value; a[k] = o[k]; });
}

// One Stockham stage of compile-time radix R over the whole tile: every thread takes butterflies (j, q, pencil p), holds
// the R inputs in registers, transforms them with the in-register DFT of fft_core.cuh (or the prime butterfly above) and
// stores the R outputs multiplied by w_n^{jk}.  Not inlined: one copy per (precision, radix, direction) serves all five kernels.
template <typename T, int R, bool INV>
__device__ __noinline__ void gen_stage(const cx<T> *x, cx<T> *y, const cx<T> *tw, int S, int P, int n, int s, int tid) {
    const int PP = gen_pitch(P), m = n / R, nbf = S / R, wn = S / n, istride = s * m * PP, ostride = s * PP;
    const int lgP = 31 - __clz(P);                   // P is a power of two
    const GenDiv by_s(s);
    for (int idx = tid; idx < nbf * P; idx += GEN_NT) {
        const int p = idx & (P - 1), b = idx >> lgP, j = by_s.div(b), q = b - j * s;
        cx<T> a[R];
        const cx<T> *src = x + (q + s * j) * PP + p;
        static_for<R>([&](auto rc) { constexpr int r = decltype(rc)::value; a[r] = src[r * istride]; });
        if constexpr (R == 11 || R == 13) gen_dft_prime<T, R, INV>(a, tw, S / R);   // radix 7 has literal twiddles in fft_core.cuh
        else dft<T, R, INV>(a);
        cx<T> *dst = y + (q + s * R * j) * PP + p;
        dst[0] = a[0];
        if (m == 1) {            // last stage: every w_n^{jk} is 1
            static_for<R - 1>([&](auto kc) { constexpr int k = decltype(kc)::value + 1; dst[k * ostride] = a[k]; });
        } else {
            static_for<R - 1>([&](auto kc) {
                constexpr int k = decltype(kc)::value + 1;
                dst[k * ostride] = a[k] * gen_w(tw, wn * j * k, INV);        // j k < n, so wn j k < S
            });
        }
    }
}

// Any other radix (primes from 17 up): one output per thread per step, the R-term sum read from shared memory.
template <typename T>
__device__ __noinline__ void gen_stage_any(const cx<T> *x, cx<T> *y, const cx<T> *tw, int S, int P, int n, int s, int R, bool inv, int tid) {
    const int PP = gen_pitch(P), m = n / R, wr = S / R, wn = S / n;
    const int lgP = 31 - __clz(P);
    for (int idx = tid; idx < S * P; idx += GEN_NT) {
        const int p = idx & (P - 1), e = idx >> lgP;   // output element e = q + s (R j + k)
        const int q = e % s, t = e / s, k = t % R, j = t / R;
        const cx<T> *src = x + (q + s * j) * PP + p;
        const int stride = s * m * PP;
        T ar = 0, ai = 0;
        int wi = 0;
        const int step = (int)(((long long)wr * k) % S);
        for (int r = 0; r < R; ++r) {
            const cx<T> a = src[r * stride], w = gen_w(tw, wi, inv);
            ar += a.re * w.re - a.im * w.im;
            ai += a.re * w.im + a.im * w.re;
            wi += step; if (wi >= S) wi -= S;
        }
        const cx<T> w = gen_w(tw, wn * j * k, inv);     // j k < n, so wn j k < S
        y[e * PP + p] = mk<T>(ar * w.re - ai * w.im, ar * w.im + ai * w.re);
    }
}

template <typename T, bool INV>
PF_HD void gen_stage_dispatch(const cx<T> *x, cx<T> *y, const cx<T> *tw, int S, int P, int n, int s, int R, int tid) {
    switch (R) {
        case 2: gen_stage<T, 2, INV>(x, y, tw, S, P, n, s, tid); break;
        case 3: gen_stage<T, 3, INV>(x, y, tw, S, P, n, s, tid); break;
        case 4: gen_stage<T, 4, INV>(x, y, tw, S, P, n, s, tid); break;
        case 5: gen_stage<T, 5, INV>(x, y, tw, S, P, n, s, tid); break;
        case 6: gen_stage<T, 6, INV>(x, y, tw, S, P, n, s, tid); break;
        case 7: gen_stage<T, 7, INV>(x, y, tw, S, P, n, s, tid); break;
        case 8: gen_stage<T, 8, INV>(x, y, tw, S, P, n, s, tid); break;
        case 10: gen_stage<T, 10, INV>(x, y, tw, S, P, n, s, tid); break;
        case 11: gen_stage<T, 11, INV>(x, y, tw, S, P, n, s, tid); break;
        case 12: gen_stage<T, 12, INV>(x, y, tw, S, P, n, s, tid); break;
        case 13: gen_stage<T, 13, INV>(x, y, tw, S, P, n, s, tid); break;
        case 14: gen_stage<T, 14, INV>(x, y, tw, S, P, n, s, tid); break;
        case 15: gen_stage<T, 15, INV>(x, y, tw, S, P, n, s, tid); break;
        case 16: gen_stage<T, 16, INV>(x, y, tw, S, P, n, s, tid); break;
        default: gen_stage_any<T>(x, y, tw, S, P, n, s, R, INV, tid); break;
    }
}

// The Stockham pass sequence over the tile in x (the function returns the buffer that holds the result); the transform
// length is gen_L (= gen_S, or the convolution length M of the Bluestein path).
template <typename T>
PF_HD cx<T> *gen_fft(cx<T> *x, cx<T> *y, const cx<T> *tw, const PassParams &prm, bool inv, int tid) {
    const int L = prm.gen_L, P = prm.gen_P;
    int n = L, s = 1;
    for (int f = 0; f < prm.gen_nfac; ++f) {
        const int R = prm.gen_fac[f];
        if (inv) gen_stage_dispatch<T, true>(x, y, tw, L, P, n, s, R, tid);
        else gen_stage_dispatch<T, false>(x, y, tw, L, P, n, s, R, tid);
        __syncthreads();
        cx<T> *tmp = x; x = y; y = tmp;
        n /= R; s *= R;
    }
    return x;
}

// Length-S DFT of every pencil of the tile.  Smooth lengths: the Stockham passes directly.  Lengths with a prime factor
// >= 17 (gen_blue): Bluestein's chirp-z -- with c_n = exp(-i pi n^2 / S),  n k = (n^2 + k^2 - (k - n)^2) / 2 gives
//     X_k = c_k  sum_n (x_n c_n) conj(c_{k-n}),
// a cyclic convolution of length M >= 2S - 1 done with two smooth length-M transforms: chirp[n] = c_n and
// bspec = FFT_M(conj c, wrapped) / M come from the plan (host, long double); the inverse DFT conjugates both.
template <typename T>
PF_HD cx<T> *gen_transform(cx<T> *x, cx<T> *y, const cx<T> *tw, const PassParams &prm, bool inv, int tid) {
    if (!prm.gen_blue) return gen_fft<T>(x, y, tw, prm, inv, tid);
    const int S = prm.gen_S, L = prm.gen_L, P = prm.gen_P, PP = gen_pitch(P), lgP = 31 - __clz(P);
    const cx<T> *chirp = reinterpret_cast<const cx<T> *>(prm.chirp), *bspec = reinterpret_cast<const cx<T> *>(prm.bspec);
    for (int idx = tid; idx < L * P; idx += GEN_NT) {
        const int p = idx & (P - 1), n = idx >> lgP;
        cx<T> v = mk<T>((T)0, (T)0);
        if (n < S) { const cx<T> c = chirp[n]; v = x[n * PP + p] * (inv ? conj(c) : c); }
        x[n * PP + p] = v;
    }
    __syncthreads();
    cx<T> *r = gen_fft<T>(x, y, tw, prm, false, tid);
    cx<T> *o = (r == x) ? y : x;
    for (int idx = tid; idx < L * P; idx += GEN_NT) {
        const int p = idx & (P - 1), k = idx >> lgP;
        const cx<T> b = bspec[k];
        r[k * PP + p] = r[k * PP + p] * (inv ? conj(b) : b);
    }
    __syncthreads();
    r = gen_fft<T>(r, o, tw, prm, true, tid);
    for (int idx = tid; idx < S * P; idx += GEN_NT) {
        const int p = idx & (P - 1), k = idx >> lgP;
        const cx<T> c = chirp[k];
        r[k * PP + p] = r[k * PP + p] * (inv ? conj(c) : c);
    }
    __syncthreads();
    return r;
}

template <typename T, int KIND>
__global__ void __launch_bounds__(GEN_NT, 2) generic_pass_kernel(const PassParams prm) {
    extern __shared__ __align__(16) unsigned char pf_smem[];
    const int S = prm.gen_S, L = prm.gen_L, P = prm.gen_P, PP = gen_pitch(P), tid = threadIdx.x;
    const int H = S / 2 + 1;
    const bool pruned = prm.gen_pruned != 0;
    cx<T> *b0 = reinterpret_cast<cx<T> *>(pf_smem), *b1 = b0 + (size_t)L * PP, *tw = b1 + (size_t)L * PP;
    pdl_launch_dependents();
    { const cx<T> *tab = reinterpret_cast<const cx<T> *>(prm.tw); for (int i = tid; i < L; i += GEN_NT) tw[i] = tab[i]; }
    pdl_wait_prior_grid();
    __syncthreads();
    const int n_half = pruned ? S / 2 : S;      // points that exist on the un-padded side of this pass
    const int lgP = 31 - __clz(P);              // P is a power of two
    const GenDiv by_S(S), by_half(n_half);

    for (int tile = blockIdx.x; tile < prm.n_tiles; tile += gridDim.x) {
        const int bi = tile / prm.n_tiles1, tl = tile - bi * prm.n_tiles1;
        const int g = tl / prm.tiles_per_g, p0 = (tl % prm.tiles_per_g) * P;
        const int ncols = prm.n_p - p0 < P ? prm.n_p - p0 : P;
        cx<T> *x = b0, *y = b1;

        // ---------------- load (spread: the zero half is generated here)
        if constexpr (KIND == KIND_F1) {            // two real pencils adjacent in x -> one complex pencil
            const T *src = (prm.use_list == 1 ? reinterpret_cast<const T *>(prm.blist[bi]) : reinterpret_cast<const T *>(prm.in) + bi * prm.bs_in) + g * prm.gs_in;
            for (int idx = tid; idx < S * P; idx += GEN_NT) {
                const int q = idx & (P - 1), n = idx >> lgP;
                cx<T> v = mk<T>((T)0, (T)0);
                if (n < n_half && q < ncols) {
                    const long long xr = 2LL * (p0 + q);
                    v.re = src[n * prm.ns_in + xr * prm.ps_in];
                    if (xr + 1 < prm.gen_nreal) v.im = src[n * prm.ns_in + (xr + 1) * prm.ps_in];
                }
                x[n * PP + q] = v;
            }
        } else if constexpr (KIND == KIND_I1) {     // Z_k = A_k + i B_k,  Z_{S-k} = conj A_k + i conj B_k
            const cx<T> *src = pass_in<T>(prm, bi) + g * prm.gs_in;
            for (int idx = tid; idx < H * P; idx += GEN_NT) {
                const int q = idx & (P - 1), k = idx >> lgP;
                cx<T> a = mk<T>((T)0, (T)0), b = a;
                if (q < ncols) {
                    const long long xr = 2LL * (p0 + q);
                    a = src[k * prm.ns_in + xr * prm.ps_in];
                    if (xr + 1 < prm.gen_nreal) b = src[k * prm.ns_in + (xr + 1) * prm.ps_in];
                }
                x[k * PP + q] = mk<T>(a.re - b.im, a.im + b.re);
                if (k > 0 && S - k >= H) x[(S - k) * PP + q] = mk<T>(a.re + b.im, b.re - a.im);
            }
        } else {
            const cx<T> *src = pass_in<T>(prm, bi) + g * prm.gs_in + p0 * prm.ps_in;
            const int n_in = (KIND == KIND_I2) ? S : n_half;
            const bool lanes_p = prm.gen_lanes_p != 0;
            for (int idx = tid; idx < S * P; idx += GEN_NT) {
                int n, p;
                if (lanes_p) { p = idx & (P - 1); n = idx >> lgP; } else { p = by_S.div(idx); n = idx - p * S; }
                x[n * PP + p] = (n < n_in && p < ncols) ? src[n * prm.ns_in + p * prm.ps_in] : mk<T>((T)0, (T)0);
            }
        }
        __syncthreads();

        // ---------------- transform(s)
        constexpr bool FIRST_INV = KIND == KIND_I2 || KIND == KIND_I1;
        cx<T> *r = gen_transform<T>(x, y, tw, prm, FIRST_INV, tid);
        cx<T> *o = (r == b0) ? b1 : b0;
        if constexpr (KIND == KIND_F3) {            // V^F = K^F rho^F (Eq. 3), then straight back
            const bool lanes_p = prm.gen_lanes_p != 0;
            const long long gk = g + prm.k_g0;   // plane chunks: position in the whole grid
            const long long kbase = lanes_p ? gk * S * prm.n_p + p0 : (gk * prm.n_p + p0) * S;
            for (int idx = tid; idx < S * P; idx += GEN_NT) {
                int k, p;
                if (lanes_p) { p = idx & (P - 1); k = idx >> lgP; } else { p = by_S.div(idx); k = idx - p * S; }
                if (p < ncols) {
                    const long long ki = kbase + (lanes_p ? (long long)k * prm.n_p + p : (long long)p * S + k);
                    const cx<T> v = r[k * PP + p];
                    if (prm.gen_kcplx) r[k * PP + p] = v * reinterpret_cast<const cx<T> *>(prm.kint)[ki];
                    else r[k * PP + p] = scale(v, reinterpret_cast<const T *>(prm.kint)[ki]);
                }
            }
            __syncthreads();
            r = gen_transform<T>(r, o, tw, prm, true, tid);
        }

        // ---------------- store (compactification: only the lower half leaves the chip)
        if constexpr (KIND == KIND_F1) {            // A = (Z_k + conj Z_{S-k}) / 2,  B = -i (Z_k - conj Z_{S-k}) / 2,  k <= S/2
            cx<T> *dst = pass_out<T>(prm, bi) + g * prm.gs_out;
            for (int idx = tid; idx < H * P; idx += GEN_NT) {
                const int q = idx & (P - 1), k = idx >> lgP;
                if (q < ncols) {
                    const cx<T> zk = r[k * PP + q], zp = r[((S - k) % S) * PP + q];
                    const T hf = (T)0.5;
                    const long long xr = 2LL * (p0 + q);
                    dst[k * prm.ns_out + xr * prm.ps_out] = mk<T>(hf * (zk.re + zp.re), hf * (zk.im - zp.im));
                    if (xr + 1 < prm.gen_nreal) dst[k * prm.ns_out + (xr + 1) * prm.ps_out] = mk<T>(hf * (zk.im + zp.im), hf * (zp.re - zk.re));
                }
            }
        } else if constexpr (KIND == KIND_I1) {     // real part -> pencil 2q, imaginary part -> pencil 2q + 1
            T *dst = (prm.use_list == 2 ? reinterpret_cast<T *>(const_cast<void *>(prm.blist[bi])) : reinterpret_cast<T *>(prm.out) + bi * prm.bs_out) + g * prm.gs_out;
            for (int idx = tid; idx < n_half * P; idx += GEN_NT) {
                const int q = idx & (P - 1), n = idx >> lgP;
                if (q < ncols) {
                    const cx<T> v = r[n * PP + q];
                    const long long xr = 2LL * (p0 + q);
                    dst[n * prm.ns_out + xr * prm.ps_out] = v.re;
                    if (xr + 1 < prm.gen_nreal) dst[n * prm.ns_out + (xr + 1) * prm.ps_out] = v.im;
                }
            }
        } else {
            cx<T> *dst = pass_out<T>(prm, bi) + g * prm.gs_out + p0 * prm.ps_out;
            const int n_out = (KIND == KIND_F2) ? S : n_half;
            const bool lanes_p = prm.gen_lanes_p != 0;
            for (int idx = tid; idx < n_out * P; idx += GEN_NT) {
                int n, p;
                if (lanes_p) { p = idx & (P - 1); n = idx >> lgP; } else { p = (n_out == S ? by_S : by_half).div(idx); n = idx - p * n_out; }
                if (p < ncols) dst[n * prm.ns_out + p * prm.ps_out] = r[n * PP + p];
            }
        }
        __syncthreads();
    }
}

// K^F re-layout for the generic F3 kernel (the kernel is transposed once): natural order of the pass,
//   lanes along pencils:   kint[(g S_c + k_c) n_p + pp]        lanes along the transform:   kint[(g n_p + pp) S_c + k_c]
// pre-multiplied by 1 / (S_x S_y S_z).  cplx: the caller's array holds complex values and the half not passed is the
// Hermitian image K^F(-k) = conj K^F(k) (a real kernel K without inversion symmetry).
struct GenericRelayoutParams {
    int S, n_p, lanes_p, cplx;
    int a_axis, c_axis;
    int sx, sy, sz;
    long long total;      // points (not reals)
    double scale;
};

template <typename T>
__global__ void generic_relayout_kernel(const T *__restrict__ kuser, T *__restrict__ kint, const GenericRelayoutParams q) {
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < q.total; idx += (long long)gridDim.x * blockDim.x) {
        long long g, kc, pp;
        if (q.lanes_p) { pp = idx % q.n_p; kc = (idx / q.n_p) % q.S; g = idx / ((long long)q.n_p * q.S); }
        else { kc = idx % q.S; pp = (idx / q.S) % q.n_p; g = idx / ((long long)q.n_p * q.S); }
        long long f[3];
        f[3 - q.a_axis - q.c_axis] = pp; f[q.c_axis] = kc; f[q.a_axis] = g;
        long long kx = f[0], ky = f[1], kz = f[2];
        const int hx = q.sx / 2 + 1;
        bool mirrored = false;
        if (kx > q.sx / 2) { kx = q.sx - kx; ky = (q.sy - ky) % q.sy; kz = (q.sz - kz) % q.sz; mirrored = true; }
        const long long u = (kz * q.sy + ky) * hx + kx;
        if (q.cplx) {
            kint[2 * idx] = (T)((double)kuser[2 * u] * q.scale);
            kint[2 * idx + 1] = (T)((double)kuser[2 * u + 1] * (mirrored ? -q.scale : q.scale));
        } else {
            kint[idx] = (T)((double)kuser[u] * q.scale);
        }
    }
}

}  // namespace pfft
