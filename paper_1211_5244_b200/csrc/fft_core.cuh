// fft_core.cuh -- in-register building blocks of the customised FFT:
// complex arithmetic, compile-time twiddles, small DFTs of radix 2..32 (factors 2, 3, 5, 7) held entirely in one
// thread's registers, and the two "pruned" variants that implement the paper's spread /
// compactification without ever touching the zero half:
//   * dft_pruned_in  : DFT of a length-R sequence whose upper half is zero   (spread,  PAPER.md:53)
//   * dft_pruned_out : DFT of a length-R sequence keeping only outputs n<R/2 (compactification)
#pragma once

#include <cstddef>
#include <utility>

#include "twiddle_consts.cuh"

#define PF_HD __device__ __forceinline__          // device code only: there is no host path
#define PF_CE __host__ __device__ constexpr       // compile-time helpers (twiddle literals, geometry)

namespace pfft {

// ------------------------------------------------------------------ complex number
template <typename T>
struct alignas(2 * sizeof(T)) cx {
    T re, im;
};

template <typename T> PF_HD cx<T> mk(T re, T im) { cx<T> r; r.re = re; r.im = im; return r; }
template <typename T> PF_HD cx<T> operator+(cx<T> a, cx<T> b) { return mk<T>(a.re + b.re, a.im + b.im); }
template <typename T> PF_HD cx<T> operator-(cx<T> a, cx<T> b) { return mk<T>(a.re - b.re, a.im - b.im); }
template <typename T> PF_HD cx<T> operator*(cx<T> a, cx<T> b) {
    return mk<T>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re);
}
template <typename T> PF_HD cx<T> scale(cx<T> a, T s) { return mk<T>(a.re * s, a.im * s); }
template <typename T> PF_HD cx<T> conj(cx<T> a) { return mk<T>(a.re, -a.im); }
template <typename T> PF_HD cx<T> mul_conj(cx<T> a, cx<T> w) {  // a * conj(w)
    return mk<T>(a.re * w.re + a.im * w.im, a.im * w.re - a.re * w.im);
}
// multiply by -i (forward quarter turn) or +i
template <typename T> PF_HD cx<T> mul_mi(cx<T> a) { return mk<T>(a.im, -a.re); }
template <typename T> PF_HD cx<T> mul_pi(cx<T> a) { return mk<T>(-a.im, a.re); }

// ------------------------------------------------------------------ streaming global accesses
// Data that is touched once per solve (rho, K^F, V, and the last read of an intermediate) is
// loaded / stored with the evict-first policy (ld.global.cs / st.global.cs) so that it does not
// push the intermediates A1 / A2, which ARE reused by the next pass, out of the 126 MB L2.
PF_HD cx<double> ld_stream(const cx<double> *p) {
    const double2 v = __ldcs(reinterpret_cast<const double2 *>(p));
    return mk<double>(v.x, v.y);
}
PF_HD cx<float> ld_stream(const cx<float> *p) {
    const float2 v = __ldcs(reinterpret_cast<const float2 *>(p));
    return mk<float>(v.x, v.y);
}
PF_HD double ld_stream(const double *p) {
    return __ldcs(p);
}
PF_HD float ld_stream(const float *p) {
    return __ldcs(p);
}
PF_HD void st_stream(cx<double> *p, cx<double> v) {
    __stcs(reinterpret_cast<double2 *>(p), make_double2(v.re, v.im));
}
PF_HD void st_stream(cx<float> *p, cx<float> v) {
    __stcs(reinterpret_cast<float2 *>(p), make_float2(v.re, v.im));
}
// Two complex values adjacent in memory as ONE access: 256-bit LDG/STG in fp64 (new on sm_100), 128-bit in fp32.
// p must be aligned to the size of the pair.
PF_HD void st_pair(cx<double> *p, cx<double> a, cx<double> b) {
    asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(a.re), "d"(a.im), "d"(b.re), "d"(b.im) : "memory");
}
PF_HD void st_pair(cx<float> *p, cx<float> a, cx<float> b) {
    *reinterpret_cast<float4 *>(p) = make_float4(a.re, a.im, b.re, b.im);
}
PF_HD void ld_pair_stream(const cx<double> *p, cx<double> &a, cx<double> &b) {
    asm volatile("ld.global.cs.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(a.re), "=d"(a.im), "=d"(b.re), "=d"(b.im) : "l"(p));
}
PF_HD void ld_pair_stream(const cx<float> *p, cx<float> &a, cx<float> &b) {
    const float4 v = __ldcs(reinterpret_cast<const float4 *>(p));
    a = mk<float>(v.x, v.y); b = mk<float>(v.z, v.w);
}
template <bool STREAM, typename E> PF_HD E ld_hint(const E *p) {
    if constexpr (STREAM) return ld_stream(p); else return *p;
}
template <bool STREAM, typename E> PF_HD void st_hint(E *p, E v) {
    if constexpr (STREAM) st_stream(p, v); else *p = v;
}

// ------------------------------------------------------------------ compile-time loops
template <int... Is, typename F>
PF_HD void static_for_impl(std::integer_sequence<int, Is...>, F &&f) {
    (f(std::integral_constant<int, Is>{}), ...);
}
template <int N, typename F>
PF_HD void static_for(F &&f) {
    static_for_impl(std::make_integer_sequence<int, N>{}, static_cast<F &&>(f));
}

// ------------------------------------------------------------------ compile-time twiddles
// cos/sin(2 pi m / R) for R | 480, reduced to the first octant of a 61-entry literal table.
PF_CE double oct_cos(int j) { constexpr double t[61] = {PFFT_OCT_COS_LIST}; return t[j]; }
PF_CE double oct_sin(int j) { constexpr double t[61] = {PFFT_OCT_SIN_LIST}; return t[j]; }

PF_CE double cos480(int j) {  // j in [0, 480)
    if (j > 240) j = 480 - j;               // cos(-x) = cos(x)
    bool neg = false;
    if (j > 120) { j = 240 - j; neg = true; }  // cos(pi - x) = -cos(x)
    double v = (j <= 60) ? oct_cos(j) : oct_sin(120 - j);
    if (j == 120) v = 0.0;
    return neg ? -v : v;
}
PF_CE double sin480(int j) {  // j in [0, 480)
    bool neg = false;
    if (j > 240) { j = 480 - j; neg = true; }  // sin(-x) = -sin(x)
    if (j > 120) j = 240 - j;                   // sin(pi - x) = sin(x)
    double v = (j <= 60) ? oct_sin(j) : oct_cos(120 - j);
    if (j == 0 || j == 240) v = 0.0;
    return neg ? -v : v;
}
PF_CE bool divides480(int R) { return R > 0 && 480 % R == 0; }
// cos/sin(2 pi m / R) for R | 28 (radices 7, 14, 28), reduced to the first quadrant of an 8-entry literal table.
PF_CE double q28_cos(int j) { constexpr double t[8] = {PFFT_R28_COS_LIST}; return t[j]; }
PF_CE double q28_sin(int j) { constexpr double t[8] = {PFFT_R28_SIN_LIST}; return t[j]; }
PF_CE double cos28(int j) {  // j in [0, 28)
    if (j > 14) j = 28 - j;
    return j <= 7 ? q28_cos(j) : -q28_cos(14 - j);
}
PF_CE double sin28(int j) {  // j in [0, 28)
    bool neg = false;
    if (j > 14) { j = 28 - j; neg = true; }
    const double v = j <= 7 ? q28_sin(j) : q28_sin(14 - j);
    return neg ? -v : v;
}
PF_CE bool divides28(int R) { return R > 0 && 28 % R == 0; }
PF_CE bool literal_radix(int R) { return divides480(R) || divides28(R); }
// real / imaginary part of exp(-2 pi i m / R)   (forward sign)
PF_CE double tw_re(int m, int R) {
    const int j = ((m % R) + R) % R;
    return divides480(R) ? cos480(j * (480 / R)) : cos28(j * (28 / R));
}
PF_CE double tw_im(int m, int R) {
    const int j = ((m % R) + R) % R;
    return divides480(R) ? -sin480(j * (480 / R)) : -sin28(j * (28 / R));
}

// a * exp(-/+ 2 pi i M / R) with M, R compile-time: trivial cases cost no multiply.
template <int M_, int R, bool INV, typename T>
PF_HD cx<T> mul_tw(cx<T> a) {
    static_assert(literal_radix(R), "radix must divide 480 or 28");
    constexpr int M = ((M_ % R) + R) % R;
    if constexpr (M == 0) {
        return a;
    } else if constexpr (4 * M == R) {
        return INV ? mul_pi(a) : mul_mi(a);
    } else if constexpr (2 * M == R) {
        return mk<T>(-a.re, -a.im);
    } else if constexpr (4 * M == 3 * R) {
        return INV ? mul_mi(a) : mul_pi(a);
    } else if constexpr (8 * M == R || 8 * M == 3 * R || 8 * M == 5 * R || 8 * M == 7 * R) {
        // (+-1 +- i)/sqrt(2): two adds and two multiplies
        constexpr T h = (T)0.70710678118654752440084436210484903928;
        constexpr double c = tw_re(M, R), s = INV ? -tw_im(M, R) : tw_im(M, R);
        // result = (c + i s)(re + i im) with |c| = |s| = h
        const T p = a.re - a.im, q = a.re + a.im;  // re*1 - im*1 ; re*1 + im*1
        if constexpr (c > 0 && s > 0) return mk<T>(h * p, h * q);         //  (1+i)/r2
        else if constexpr (c > 0 && s < 0) return mk<T>(h * q, -(h * p)); //  (1-i)/r2
        else if constexpr (c < 0 && s > 0) return mk<T>(-(h * q), h * p); // (-1+i)/r2
        else return mk<T>(-(h * p), -(h * q));                            // (-1-i)/r2
    } else {
        constexpr T c = (T)tw_re(M, R);
        constexpr T s = (T)(INV ? -tw_im(M, R) : tw_im(M, R));
        return mk<T>(a.re * c - a.im * s, a.re * s + a.im * c);
    }
}

// ------------------------------------------------------------------ small DFTs (natural order in, natural order out)
// X[k] = sum_n x[n] exp(-/+ 2 pi i n k / R)   (INV: + sign, unnormalised)
template <typename T, int R, bool INV> struct Dft;

template <typename T, bool INV> struct Dft<T, 1, INV> { static PF_HD void run(cx<T> *) {} };

template <typename T, bool INV> struct Dft<T, 2, INV> {
    static PF_HD void run(cx<T> *x) {
        const cx<T> a = x[0], b = x[1];
        x[0] = a + b; x[1] = a - b;
    }
};

template <typename T, bool INV> struct Dft<T, 3, INV> {
    static PF_HD void run(cx<T> *x) {
        constexpr T s3 = (T)0.86602540378443864676372317075293618347;  // sin(2 pi/3)
        const cx<T> t1 = x[1] + x[2];
        const cx<T> t2 = mk<T>(x[0].re - (T)0.5 * t1.re, x[0].im - (T)0.5 * t1.im);
        const cx<T> d = x[1] - x[2];
        // forward: X1 = t2 - i s3 d ; X2 = t2 + i s3 d
        const cx<T> t3 = INV ? mk<T>(-s3 * d.im, s3 * d.re) : mk<T>(s3 * d.im, -(s3 * d.re));
        x[0] = x[0] + t1; x[1] = t2 + t3; x[2] = t2 - t3;
    }
};

template <typename T, bool INV> struct Dft<T, 4, INV> {
    static PF_HD void run(cx<T> *x) {
        const cx<T> a = x[0] + x[2], b = x[0] - x[2], c = x[1] + x[3], d = x[1] - x[3];
        const cx<T> jd = INV ? mul_pi(d) : mul_mi(d);  // forward: -i d
        x[0] = a + c; x[1] = b + jd; x[2] = a - c; x[3] = b - jd;
    }
};

template <typename T, bool INV> struct Dft<T, 5, INV> {
    static PF_HD void run(cx<T> *x) {
        constexpr T c1 = (T)0.30901699437494742410229341718281905886;   // cos(2 pi/5)
        constexpr T c2 = (T)-0.80901699437494742410229341718281905886;  // cos(4 pi/5)
        constexpr T s1 = (T)0.95105651629515357211643933337938214340;   // sin(2 pi/5)
        constexpr T s2 = (T)0.58778525229247312916870595463907276860;   // sin(4 pi/5)
        const cx<T> a1 = x[1] + x[4], b1 = x[1] - x[4], a2 = x[2] + x[3], b2 = x[2] - x[3];
        const cx<T> m1 = mk<T>(x[0].re + c1 * a1.re + c2 * a2.re, x[0].im + c1 * a1.im + c2 * a2.im);
        const cx<T> m2 = mk<T>(x[0].re + c2 * a1.re + c1 * a2.re, x[0].im + c2 * a1.im + c1 * a2.im);
        const cx<T> u1 = mk<T>(s1 * b1.re + s2 * b2.re, s1 * b1.im + s2 * b2.im);
        const cx<T> u2 = mk<T>(s2 * b1.re - s1 * b2.re, s2 * b1.im - s1 * b2.im);
        // forward: X1 = m1 - i u1, X4 = m1 + i u1, X2 = m2 - i u2, X3 = m2 + i u2
        const cx<T> v1 = INV ? mul_pi(u1) : mul_mi(u1);
        const cx<T> v2 = INV ? mul_pi(u2) : mul_mi(u2);
        x[0] = x[0] + a1 + a2;
        x[1] = m1 + v1; x[4] = m1 - v1; x[2] = m2 + v2; x[3] = m2 - v2;
    }
};

// radix 7: a_j = x_j + x_{7-j}, b_j = x_j - x_{7-j};  X_k, X_{7-k} = x_0 + sum_j cos(2 pi jk/7) a_j  -/+  i sum_j sin(2 pi jk/7) b_j
template <typename T, bool INV> struct Dft<T, 7, INV> {
    static PF_HD void run(cx<T> *x) {
        constexpr T c1 = (T)0.6234898018587335305250048840042398106323;    // cos(2 pi/7)
        constexpr T c2 = (T)-0.2225209339563144042889025644967947594664;   // cos(4 pi/7)
        constexpr T c3 = (T)-0.9009688679024191262361023195074450511659;   // cos(6 pi/7)
        constexpr T s1 = (T)0.7818314824680298087084445266740577502323;    // sin(2 pi/7)
        constexpr T s2 = (T)0.9749279121818236070181316829939312172328;    // sin(4 pi/7)
        constexpr T s3 = (T)0.43388373911755812047576833284835875461;      // sin(6 pi/7)
        const cx<T> a1 = x[1] + x[6], b1 = x[1] - x[6], a2 = x[2] + x[5], b2 = x[2] - x[5], a3 = x[3] + x[4], b3 = x[3] - x[4];
        // cos(2 pi jk/7): k = 1: c1 c2 c3;  k = 2: c2 c3 c1;  k = 3: c3 c1 c2.   sin: k = 1: s1 s2 s3;  k = 2: s2 -s3 -s1;  k = 3: s3 -s1 s2
        const cx<T> m1 = mk<T>(x[0].re + c1 * a1.re + c2 * a2.re + c3 * a3.re, x[0].im + c1 * a1.im + c2 * a2.im + c3 * a3.im);
        const cx<T> m2 = mk<T>(x[0].re + c2 * a1.re + c3 * a2.re + c1 * a3.re, x[0].im + c2 * a1.im + c3 * a2.im + c1 * a3.im);
        const cx<T> m3 = mk<T>(x[0].re + c3 * a1.re + c1 * a2.re + c2 * a3.re, x[0].im + c3 * a1.im + c1 * a2.im + c2 * a3.im);
        const cx<T> u1 = mk<T>(s1 * b1.re + s2 * b2.re + s3 * b3.re, s1 * b1.im + s2 * b2.im + s3 * b3.im);
        const cx<T> u2 = mk<T>(s2 * b1.re - s3 * b2.re - s1 * b3.re, s2 * b1.im - s3 * b2.im - s1 * b3.im);
        const cx<T> u3 = mk<T>(s3 * b1.re - s1 * b2.re + s2 * b3.re, s3 * b1.im - s1 * b2.im + s2 * b3.im);
        // forward: X_k = m_k - i u_k, X_{7-k} = m_k + i u_k
        const cx<T> v1 = INV ? mul_pi(u1) : mul_mi(u1);
        const cx<T> v2 = INV ? mul_pi(u2) : mul_mi(u2);
        const cx<T> v3 = INV ? mul_pi(u3) : mul_mi(u3);
        x[0] = x[0] + a1 + a2 + a3;
        x[1] = m1 + v1; x[6] = m1 - v1; x[2] = m2 + v2; x[5] = m2 - v2; x[3] = m3 + v3; x[4] = m3 - v3;
    }
};

// first factor A of the Cooley-Tukey split R = A * B used for composite radices
PF_CE int split_a(int R) {
    return R == 6 ? 2 : R == 8 ? 2 : R == 10 ? 2 : R == 12 ? 3 : R == 14 ? 2 : R == 15 ? 3 : R == 16 ? 4 : R == 20 ? 4
         : R == 24 ? 3 : R == 28 ? 4 : R == 32 ? 4 : 0;
}

// Composite: n = n1 + B n2, k = k2 + A k1;  X[k2 + A k1] = sum_n1 w_B^{n1 k1} [ w_R^{n1 k2} sum_n2 x[n1 + B n2] w_A^{n2 k2} ]
template <typename T, int R, bool INV> struct Dft {
    static constexpr int A = split_a(R), B = R / A;
    static_assert(A > 1 && A * B == R, "unsupported in-register radix");
    static PF_HD void run(cx<T> *x) {
        cx<T> y[R];  // y[n1 * A + k2]
        static_for<B>([&](auto n1c) {
            constexpr int n1 = decltype(n1c)::value;
            cx<T> u[A];
            static_for<A>([&](auto n2c) { constexpr int n2 = decltype(n2c)::value; u[n2] = x[n1 + B * n2]; });
            Dft<T, A, INV>::run(u);
            static_for<A>([&](auto k2c) {
                constexpr int k2 = decltype(k2c)::value;
                y[n1 * A + k2] = mul_tw<n1 * k2, R, INV>(u[k2]);
            });
        });
        static_for<A>([&](auto k2c) {
            constexpr int k2 = decltype(k2c)::value;
            cx<T> g[B];
            static_for<B>([&](auto n1c) { constexpr int n1 = decltype(n1c)::value; g[n1] = y[n1 * A + k2]; });
            Dft<T, B, INV>::run(g);
            static_for<B>([&](auto k1c) { constexpr int k1 = decltype(k1c)::value; x[k2 + A * k1] = g[k1]; });
        });
    }
};

template <typename T, int R, bool INV> PF_HD void dft(cx<T> *x) { Dft<T, R, INV>::run(x); }

// Spread in registers: x[0..R/2) hold data, x[R/2..R) are zeros that are never
// stored anywhere.  X[2j] = DFT_{R/2}(x)[j],  X[2j+1] = DFT_{R/2}(x[n] w_R^n)[j].
template <typename T, int R, bool INV> PF_HD void dft_pruned_in(cx<T> *x) {
    static_assert(R % 2 == 0, "pruned radix must be even");
    constexpr int Hh = R / 2;
    cx<T> e[Hh], o[Hh];
    static_for<Hh>([&](auto nc) {
        constexpr int n = decltype(nc)::value;
        e[n] = x[n];
        o[n] = mul_tw<n, R, INV>(x[n]);
    });
    Dft<T, Hh, INV>::run(e);
    Dft<T, Hh, INV>::run(o);
    static_for<Hh>([&](auto jc) {
        constexpr int j = decltype(jc)::value;
        x[2 * j] = e[j]; x[2 * j + 1] = o[j];
    });
}

// Compactification in registers: all R inputs, only outputs n < R/2 are formed:
// y[n] = DFT_{R/2}(x_even)[n] + w_R^{n} DFT_{R/2}(x_odd)[n].  Results land in x[0..R/2).
template <typename T, int R, bool INV> PF_HD void dft_pruned_out(cx<T> *x) {
    static_assert(R % 2 == 0, "pruned radix must be even");
    constexpr int Hh = R / 2;
    cx<T> e[Hh], o[Hh];
    static_for<Hh>([&](auto jc) {
        constexpr int j = decltype(jc)::value;
        e[j] = x[2 * j]; o[j] = x[2 * j + 1];
    });
    Dft<T, Hh, INV>::run(e);
    Dft<T, Hh, INV>::run(o);
    static_for<Hh>([&](auto nc) {
        constexpr int n = decltype(nc)::value;
        x[n] = e[n] + mul_tw<n, R, INV>(o[n]);
    });
}

}  // namespace pfft
