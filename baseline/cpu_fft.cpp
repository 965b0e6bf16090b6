// cpu_fft.cpp -- timed CPU baseline: the paper's customised 3D FFT Poisson solve (steps 57-71) on the host,
// the analogue of the paper's own "CPU implementation of the same method" (there with FFTW, here with a plain
// FFTW-free Stockham FFT of our own).  Reported by bench.py beside the GPU numbers -- a baseline, not a target.
//
// It is neither the product (that is the CUDA library) nor the oracle (oracle/poisson_oracle.c is the O(n^2) definition):
// it shares no code with either, and tests/test_cpu_baseline.py checks it against the oracle.
//
// Method, as in the paper: 1D FFTs only on rows that are not identically zero:
//   step 1  N_y N_z real rows along x, zero padded to S_x, real-to-complex (two rows per complex FFT), keep S_x/2+1
//   step 2  (S_x/2+1) N_c pencils along the second axis b, padded to S_b
//   step 3  (S_x/2+1) S_b pencils along the third axis c, padded to S_c; multiply by K^F (Eq. 3); inverse along c,
//           keep the first N_c
//   step 4  inverse along b, keep N_b;   step 5  inverse along x (complex-to-real), keep N_x.
// Of y and z the periodic axis is processed before the free one.  fp64, OpenMP over independent pencils.
//
// build: g++ -O3 -march=native -fcx-limited-range -fopenmp -shared -fPIC baseline/cpu_fft.cpp -o baseline/libcpu_fft.so
#include <algorithm>
#include <cmath>
#include <complex>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

using cd = std::complex<double>;

struct Fft1d {          // Stockham autosort, radices 4 / 2 / 3 / 5 and generic odd primes, unnormalised
    int S;
    std::vector<int> radices;
    std::vector<cd> w;  // exp(-2 pi i m / S)
    explicit Fft1d(int S_) : S(S_), w(S_ > 0 ? S_ : 1) {
        const long double two_pi = 6.283185307179586476925286766559005768L;
        for (int m = 0; m < S; ++m) w[m] = cd((double)cosl(two_pi * m / S), (double)-sinl(two_pi * m / S));
        int n = S;
        while (n % 4 == 0) { radices.push_back(4); n /= 4; }
        for (int p = 2; n > 1; ++p) while (n % p == 0) { radices.push_back(p); n /= p; }
    }
    // x: input (destroyed), y: scratch; returns the buffer holding the result.  inv: conjugate twiddles.
    cd *run(cd *x, cd *y, bool inv) const {
        int n = S, s = 1;
        auto W = [&](int i) { return inv ? std::conj(w[i]) : w[i]; };
        for (int R : radices) {
            const int m = n / R, wn = S / n;
            if (R == 2) {
                for (int j = 0; j < m; ++j) {
                    const cd t = W(wn * j);
                    for (int q = 0; q < s; ++q) {
                        const cd a = x[q + s * j], b = x[q + s * (j + m)];
                        y[q + s * (2 * j)] = a + b;
                        y[q + s * (2 * j + 1)] = (a - b) * t;
                    }
                }
            } else if (R == 4) {
                for (int j = 0; j < m; ++j) {
                    const cd t1 = W(wn * j), t2 = W(2 * wn * j), t3 = W(3 * wn * j);
                    for (int q = 0; q < s; ++q) {
                        const cd a = x[q + s * j], b = x[q + s * (j + m)], c = x[q + s * (j + 2 * m)], d = x[q + s * (j + 3 * m)];
                        const cd apc = a + c, amc = a - c, bpd = b + d, bmd = b - d;
                        const cd jbmd = inv ? cd(-bmd.imag(), bmd.real()) : cd(bmd.imag(), -bmd.real());   // -/+ i (b - d)
                        y[q + s * (4 * j)] = apc + bpd;
                        y[q + s * (4 * j + 1)] = (amc + jbmd) * t1;
                        y[q + s * (4 * j + 2)] = (apc - bpd) * t2;
                        y[q + s * (4 * j + 3)] = (amc - jbmd) * t3;
                    }
                }
            } else {                        // radix-R butterfly written out (R = 3, 5 and any other prime)
                const int wr = S / R;
                for (int j = 0; j < m; ++j)
                    for (int k = 0; k < R; ++k) {
                        const cd t = W(wn * j * k);
                        for (int q = 0; q < s; ++q) {
                            cd acc(0.0, 0.0);
                            for (int r = 0; r < R; ++r) acc += x[q + s * (j + m * r)] * W((int)(((long long)wr * r * k) % S));
                            y[q + s * (R * j + k)] = acc * t;
                        }
                    }
            }
            std::swap(x, y);
            n = m; s *= R;
        }
        return x;
    }
};

}  // namespace

extern "C" {

int cpu_fft_max_threads() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// rho, V: [nz][ny][nx] reals;  Kf_half: [Sz][Sy][Sx/2+1] reals (spectrum of an inversion-symmetric kernel);  bc[a] = 0 free
// (S = 2N), 1 periodic (S = N).  threads <= 0: all cores.  Returns 0, or 1 on bad arguments.
int cpu_poisson_solve(const double *rho, const double *Kf_half, double *V, const int n[3], const int bc[3], int threads) {
    if (!rho || !Kf_half || !V || !n || !bc) return 1;
    int S[3];
    for (int a = 0; a < 3; ++a) { if (n[a] <= 0) return 1; S[a] = n[a] * (bc[a] == 0 ? 2 : 1); }
    const int nx = n[0], ny = n[1], nz = n[2], Sx = S[0], Sy = S[1], Sz = S[2], H = Sx / 2 + 1;
#ifdef _OPENMP
    const int nth = threads > 0 ? threads : omp_get_max_threads();
#else
    const int nth = 1; (void)threads;
#endif
    // of y and z: periodic first, free last
    const bool y_first = !(bc[1] == 0 && bc[2] == 1);
    const Fft1d fx(Sx), fy(Sy), fz(Sz);
    const size_t a1n = (size_t)nz * ny * H;
    // after step 2 the second axis is padded: [nz][Sy][H] (y first) or [Sz][ny][H] (z first)
    const size_t a2n = y_first ? (size_t)nz * Sy * H : (size_t)Sz * ny * H;
    // workspace kept between calls (repeated solves with one kernel are the paper's usage)
    static std::vector<cd> A1, A2;
    if (A1.size() < a1n) A1.resize(a1n);
    if (A2.size() < a2n) A2.resize(a2n);
    const double scale = 1.0 / ((double)Sx * Sy * Sz);
    const int smax = std::max(Sx, std::max(Sy, Sz));

#pragma omp parallel num_threads(nth)
    {
        std::vector<cd> buf0(smax), buf1(smax);
        // ---- step 1: x, real-to-complex, two rows per transform
        const long long rows = (long long)ny * nz;
#pragma omp for schedule(static)
        for (long long rp = 0; rp < (rows + 1) / 2; ++rp) {
            const long long r0 = 2 * rp, r1 = r0 + 1;
            const double *p0 = rho + r0 * nx, *p1 = r1 < rows ? rho + r1 * nx : nullptr;
            for (int x = 0; x < nx; ++x) buf0[x] = cd(p0[x], p1 ? p1[x] : 0.0);
            for (int x = nx; x < Sx; ++x) buf0[x] = cd(0.0, 0.0);
            const cd *z = fx.run(buf0.data(), buf1.data(), false);
            cd *o0 = A1.data() + r0 * H, *o1 = p1 ? A1.data() + r1 * H : nullptr;
            for (int k = 0; k < H; ++k) {
                const cd zk = z[k], zp = std::conj(z[(Sx - k) % Sx]);
                o0[k] = 0.5 * (zk + zp);
                if (o1) o1[k] = cd(0.0, -0.5) * (zk - zp);
            }
        }
        // Steps 2-4 work on pencils that are strided in memory (element stride `es`, k fastest).  KB pencils adjacent in k
        // are gathered together, so that every 64-byte line fetched is used whole.
        constexpr int KB = 4;
        std::vector<cd> g0((size_t)KB * smax), g1((size_t)KB * smax);
        // pencil group: n_in values at src + i*es_in (zero padded to S), transform(s), n_out values to dst + i*es_out
        auto pencils = [&](const Fft1d &f, const cd *src, size_t es_in, int n_in, cd *dst, size_t es_out, int n_out, int kb,
                           bool inv, const double *kmul, size_t es_k) {
            const int S1 = f.S;
            for (int i = 0; i < n_in; ++i) for (int j = 0; j < kb; ++j) g0[(size_t)j * smax + i] = src[i * es_in + j];
            for (int j = 0; j < kb; ++j) {
                cd *a = g0.data() + (size_t)j * smax, *b = g1.data() + (size_t)j * smax;
                for (int i = n_in; i < S1; ++i) a[i] = cd(0.0, 0.0);
                cd *r = f.run(a, b, inv);
                if (kmul) {                  // step 3: K^F multiply, then straight back
                    cd *other = r == a ? b : a;
                    for (int i = 0; i < S1; ++i) r[i] *= kmul[i * es_k + j] * scale;
                    r = f.run(r, other, true);
                }
                if (r != a) std::memcpy(a, r, sizeof(cd) * (size_t)n_out);
            }
            for (int i = 0; i < n_out; ++i) for (int j = 0; j < kb; ++j) dst[i * es_out + j] = g0[(size_t)j * smax + i];
        };
        const int kgroups = (H + KB - 1) / KB;
        // ---- step 2: second axis b (y if y_first else z), padded
        if (y_first) {
#pragma omp for schedule(static) collapse(2)
            for (int z = 0; z < nz; ++z)
                for (int kg = 0; kg < kgroups; ++kg) {
                    const int k = kg * KB, kb = std::min(KB, H - k);
                    pencils(fy, A1.data() + (size_t)z * ny * H + k, H, ny, A2.data() + (size_t)z * Sy * H + k, H, Sy, kb, false, nullptr, 0);
                }
        } else {
#pragma omp for schedule(static) collapse(2)
            for (int y = 0; y < ny; ++y)
                for (int kg = 0; kg < kgroups; ++kg) {
                    const int k = kg * KB, kb = std::min(KB, H - k);
                    pencils(fz, A1.data() + (size_t)y * H + k, (size_t)ny * H, nz, A2.data() + (size_t)y * H + k, (size_t)ny * H, Sz, kb, false, nullptr, 0);
                }
        }
        // ---- step 3: third axis c forward, K^F multiply, inverse, keep the first N_c (the full spectrum never exists)
        if (y_first) {       // c = z: A2 is [nz][Sy][H]
#pragma omp for schedule(static) collapse(2)
            for (int y = 0; y < Sy; ++y)
                for (int kg = 0; kg < kgroups; ++kg) {
                    const int k = kg * KB, kb = std::min(KB, H - k);
                    cd *p = A2.data() + (size_t)y * H + k;
                    pencils(fz, p, (size_t)Sy * H, nz, p, (size_t)Sy * H, nz, kb, false, Kf_half + (size_t)y * H + k, (size_t)Sy * H);
                }
        } else {             // c = y: A2 is [Sz][ny][H]
#pragma omp for schedule(static) collapse(2)
            for (int z = 0; z < Sz; ++z)
                for (int kg = 0; kg < kgroups; ++kg) {
                    const int k = kg * KB, kb = std::min(KB, H - k);
                    cd *p = A2.data() + (size_t)z * ny * H + k;
                    pencils(fy, p, H, ny, p, H, ny, kb, false, Kf_half + (size_t)z * Sy * H + k, H);
                }
        }
        // ---- step 4: inverse along b, keep N_b
        if (y_first) {
#pragma omp for schedule(static) collapse(2)
            for (int z = 0; z < nz; ++z)
                for (int kg = 0; kg < kgroups; ++kg) {
                    const int k = kg * KB, kb = std::min(KB, H - k);
                    pencils(fy, A2.data() + (size_t)z * Sy * H + k, H, Sy, A1.data() + (size_t)z * ny * H + k, H, ny, kb, true, nullptr, 0);
                }
        } else {
#pragma omp for schedule(static) collapse(2)
            for (int y = 0; y < ny; ++y)
                for (int kg = 0; kg < kgroups; ++kg) {
                    const int k = kg * KB, kb = std::min(KB, H - k);
                    pencils(fz, A2.data() + (size_t)y * H + k, (size_t)ny * H, Sz, A1.data() + (size_t)y * H + k, (size_t)ny * H, nz, kb, true, nullptr, 0);
                }
        }
        // ---- step 5: inverse along x, complex-to-real (two rows per transform), keep N_x
#pragma omp for schedule(static)
        for (long long rp = 0; rp < (rows + 1) / 2; ++rp) {
            const long long r0 = 2 * rp, r1 = r0 + 1;
            const cd *a = A1.data() + r0 * H, *b = r1 < rows ? A1.data() + r1 * H : nullptr;
            for (int k = 0; k < H; ++k) {
                const cd ak = a[k], bk = b ? b[k] : cd(0.0, 0.0);
                buf0[k] = ak + cd(0.0, 1.0) * bk;
                if (k > 0 && Sx - k >= H) buf0[Sx - k] = std::conj(ak) + cd(0.0, 1.0) * std::conj(bk);
            }
            const cd *v = fx.run(buf0.data(), buf1.data(), true);
            double *o0 = V + r0 * nx, *o1 = b ? V + r1 * nx : nullptr;
            for (int x = 0; x < nx; ++x) { o0[x] = v[x].real(); if (o1) o1[x] = v[x].imag(); }
        }
    }
    return 0;
}

}  // extern "C"
