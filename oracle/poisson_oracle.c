/*
 * poisson_oracle.c -- TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct CPU oracle for the
 * Fourier-space Poisson solve of arxiv 1211.5244 (Dugan, Genovese, Goedecker).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load
 * this file's library.  It shares no code, header, table or constant generator with the CUDA path
 * under paper_1211_5244_b200/csrc/.
 *
 * What it computes, and the passages it follows:
 *   - oracle_direct_sum*:   Eq. 2 written out as the O(N^2) sum
 *                           V[i] = sum_{i' in box} K[(i - i') mod S] rho[i'],  i in box,
 *                           with S_i = N_i * B_i (B = 1 periodic, 2 free).
 *                           On a free axis S = 2N so i - i' in [-(N-1), N-1] never aliases.
 *   - oracle_dft_axis:      the discrete Fourier transform by its definition,
 *                           X[k] = sum_j x[j] exp(-/+ 2 pi i j k / S), one axis at a time, O(S^2) per line.
 *   - oracle_kernel_spectrum: K_f = DFT3(K) by three oracle_dft_axis sweeps (K^F of Eq. 3).
 *   - oracle_kernel_spectrum_c / oracle_solve_c: the same two routines for a real kernel K WITHOUT the symmetry
 *                           K(-r) = K(r): Eq. 2 and Eq. 3 hold for any K; the spectrum is then complex
 *                           with K_f(-k) = conj K_f(k) (complex K_f; outlook PAPER.md:93).
 *   - oracle_solve:         Eq. 3 on the EXPLICITLY zero-padded grid:
 *                           pad -> DFT along each axis -> multiply by K_f -> inverse DFT along each
 *                           axis -> divide by S_x S_y S_z -> copy the physical box out.
 *                           Nothing from PAPER.md section 3 (no pruning, no R2C, no transposes).
 *
 * Readings of the paper (full table in DESIGN.md): data in the first half [0,N), zeros in [N,2N);
 * forward sign exp(-2 pi i jk/S); unnormalised forward, 1/(S_x S_y S_z) applied once; no h^3.
 *
 * Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): brute-force direct sum for all 8 BC
 * combinations, Parseval, delta -> kernel, identity kernel, shift kernel (zero fill vs wrap),
 * linearity, fully periodic plane-wave closed form, mirror symmetry, and numpy's pocketfft as a
 * test-only second opinion; the complex-spectrum routines against the same brute-force sum with kernels
 * that have no symmetry at all, all 8 BC combinations.  The paper prints no worked numerical example, so no value fixture
 * exists; the closed-form 1D-FFT-count ratios 7/12 and 2/3 are in tests/golden/.
 *
 * Arithmetic: fp64 data; twiddle table w[m] = exp(-2 pi i m / S) evaluated in long double and
 * rounded once; accumulation in double (accum_ld = 0) or long double (accum_ld = 1, used by the
 * pins to bound the oracle's own rounding).  OpenMP only parallelises over independent lines /
 * output points; the order of every sum is the textbook one (j ascending).
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef double _Complex cplx;

#define ORACLE_OK 0
#define ORACLE_EINVAL 1
#define ORACLE_ENOMEM 2

/* ---- DFT by definition along one axis of a dense C-order array dims = {d0 (slowest), d1, d2} ---- */
/* sign = -1 forward, +1 inverse (unnormalised).  In place. */
int oracle_dft_axis(cplx *a, const long long dims[3], int axis, int sign, int accum_ld)
{
    if (!a || axis < 0 || axis > 2 || (sign != 1 && sign != -1)) return ORACLE_EINVAL;
    const long long S = dims[axis];
    long long stride = 1;
    for (int d = 2; d > axis; --d) stride *= dims[d];
    long long outer = 1;
    for (int d = 0; d < axis; ++d) outer *= dims[d];
    const long long inner = stride; /* lines with the same outer index are `inner` apart by 1 */

    /* w[m] = exp(sign * 2 pi i m / S), long double evaluation, rounded once to double. */
    cplx *w = (cplx *)malloc(sizeof(cplx) * (size_t)S);
    long double *wl_re = NULL, *wl_im = NULL;
    if (!w) return ORACLE_ENOMEM;
    if (accum_ld) {
        wl_re = (long double *)malloc(sizeof(long double) * (size_t)S);
        wl_im = (long double *)malloc(sizeof(long double) * (size_t)S);
        if (!wl_re || !wl_im) { free(w); free(wl_re); free(wl_im); return ORACLE_ENOMEM; }
    }
    const long double two_pi = 6.283185307179586476925286766559005768L;
    for (long long m = 0; m < S; ++m) {
        long double ang = (long double)sign * two_pi * (long double)m / (long double)S;
        long double c = cosl(ang), s = sinl(ang);
        /* exact values on the axes, so that e.g. S = 4 has no 1e-20 residue */
        if ((4 * m) % S == 0) {
            long long q = (4 * m) / S; /* quarter turns */
            c = (q == 0) ? 1.0L : (q == 2) ? -1.0L : 0.0L;
            s = (q == 1) ? (long double)sign : (q == 3) ? -(long double)sign : 0.0L;
        }
        w[m] = (double)c + (double)s * I;
        if (accum_ld) { wl_re[m] = c; wl_im[m] = s; }
    }

    int status = ORACLE_OK;
#pragma omp parallel
    {
        cplx *line = (cplx *)malloc(sizeof(cplx) * (size_t)S);
        cplx *res = (cplx *)malloc(sizeof(cplx) * (size_t)S);
        if (!line || !res) {
#pragma omp critical
            status = ORACLE_ENOMEM;
        } else {
#pragma omp for schedule(static)
            for (long long l = 0; l < outer * inner; ++l) {
                const long long o = l / inner, in = l % inner;
                cplx *base = a + o * S * stride + in;
                for (long long j = 0; j < S; ++j) line[j] = base[j * stride];
                if (!accum_ld) {
                    for (long long k = 0; k < S; ++k) {
                        double sr = 0.0, si = 0.0;
                        long long m = 0; /* m == (j * k) mod S, kept by addition */
                        for (long long j = 0; j < S; ++j) {
                            const cplx t = w[m];
                            m += k; if (m >= S) m -= S;
                            const double xr = creal(line[j]), xi = cimag(line[j]);
                            sr += xr * creal(t) - xi * cimag(t);
                            si += xr * cimag(t) + xi * creal(t);
                        }
                        res[k] = sr + si * I;
                    }
                } else {
                    for (long long k = 0; k < S; ++k) {
                        long double sr = 0.0L, si = 0.0L;
                        long long m = 0; /* m == (j * k) mod S */
                        for (long long j = 0; j < S; ++j) {
                            const long double xr = creal(line[j]), xi = cimag(line[j]);
                            sr += xr * wl_re[m] - xi * wl_im[m];
                            si += xr * wl_im[m] + xi * wl_re[m];
                            m += k; if (m >= S) m -= S;
                        }
                        res[k] = (double)sr + (double)si * I;
                    }
                }
                for (long long k = 0; k < S; ++k) base[k * stride] = res[k];
            }
        }
        free(line);
        free(res);
    }
    free(w); free(wl_re); free(wl_im);
    return status;
}

/* ---- K_f = DFT3(K): K real [Sz][Sy][Sx]; outputs the full complex spectrum's real part and the
 * largest |imag| seen (zero up to rounding iff K(-r) = K(r)).  K^F of Eq. 3. ---- */
int oracle_kernel_spectrum(const double *K, const long long S[3] /* Sx,Sy,Sz */, double *Kf_re_full,
                           double *max_abs_imag, int accum_ld)
{
    if (!K || !S || !Kf_re_full) return ORACLE_EINVAL;
    const long long dims[3] = {S[2], S[1], S[0]};
    const long long tot = dims[0] * dims[1] * dims[2];
    cplx *a = (cplx *)malloc(sizeof(cplx) * (size_t)tot);
    if (!a) return ORACLE_ENOMEM;
    for (long long i = 0; i < tot; ++i) a[i] = K[i];
    int st = ORACLE_OK;
    for (int ax = 2; ax >= 0 && st == ORACLE_OK; --ax) st = oracle_dft_axis(a, dims, ax, -1, accum_ld);
    double mi = 0.0;
    if (st == ORACLE_OK)
        for (long long i = 0; i < tot; ++i) {
            Kf_re_full[i] = creal(a[i]);
            const double im = fabs(cimag(a[i]));
            if (im > mi) mi = im;
        }
    if (max_abs_imag) *max_abs_imag = mi;
    free(a);
    return st;
}

/* ---- K_f = DFT3(K) for a real K with no symmetry: the full complex spectrum [Sz][Sy][Sx]. ---- */
int oracle_kernel_spectrum_c(const double *K, const long long S[3] /* Sx,Sy,Sz */, cplx *Kf_full, int accum_ld)
{
    if (!K || !S || !Kf_full) return ORACLE_EINVAL;
    const long long dims[3] = {S[2], S[1], S[0]};
    const long long tot = dims[0] * dims[1] * dims[2];
    for (long long i = 0; i < tot; ++i) Kf_full[i] = K[i];
    int st = ORACLE_OK;
    for (int ax = 2; ax >= 0 && st == ORACLE_OK; --ax) st = oracle_dft_axis(Kf_full, dims, ax, -1, accum_ld);
    return st;
}

static long long wrap(long long i, long long S) { return ((i % S) + S) % S; }

/* ---- Eq. 3 on the explicitly padded grid.
 *  rho      : real [nz][ny][nx]
 *  Kf_half  : real [Sz][Sy][Sx/2+1]  (the library's data contract; numpy rfftn shape).  The other
 *             half is K_f(-k) = K_f(k) (K real in real space with a real spectrum).
 *  V        : real [nz][ny][nx]
 *  bc[a]    : 0 free (S = 2N), 1 periodic (S = N), a = x,y,z
 *  axis_order: the order in which the three forward DFT sweeps run (0 = x, 1 = y, 2 = z); the
 *             inverse sweeps run in reverse.  The result does not depend on it; it only selects
 *             which intermediates `stages` receives.
 *  stages   : optional, 6 * Sz*Sy*Sx complex: the padded array after each forward sweep (0,1,2),
 *             after the K_f multiply (3), after the first and second inverse sweeps (4,5).
 *  max_abs_imag_V: largest |Im| of the unnormalised result inside the box (should be rounding). */
static int solve_core(const double *rho, const double *Kf_half, const cplx *Kf_half_c, double *V, const long long n[3],
                      const int bc[3], const int axis_order[3], cplx *stages, double *max_abs_imag_V,
                      int accum_ld)
{
    if (!rho || (!Kf_half && !Kf_half_c) || !V || !n || !bc) return ORACLE_EINVAL;
    long long S[3];
    for (int a = 0; a < 3; ++a) {
        if (n[a] <= 0 || (bc[a] != 0 && bc[a] != 1)) return ORACLE_EINVAL;
        S[a] = n[a] * (bc[a] == 0 ? 2 : 1);
    }
    int order[3] = {0, 1, 2};
    if (axis_order) for (int a = 0; a < 3; ++a) order[a] = axis_order[a];
    const long long dims[3] = {S[2], S[1], S[0]};
    const long long tot = dims[0] * dims[1] * dims[2];
    const long long H = S[0] / 2 + 1;
    cplx *a = (cplx *)calloc((size_t)tot, sizeof(cplx));
    if (!a) return ORACLE_ENOMEM;

    /* zero padding: data in [0,N), zeros in [N,S) on every free axis */
    for (long long z = 0; z < n[2]; ++z)
        for (long long y = 0; y < n[1]; ++y)
            for (long long x = 0; x < n[0]; ++x)
                a[(z * S[1] + y) * S[0] + x] = rho[(z * n[1] + y) * n[0] + x];

    int st = ORACLE_OK;
    for (int i = 0; i < 3 && st == ORACLE_OK; ++i) {
        st = oracle_dft_axis(a, dims, 2 - order[i], -1, accum_ld); /* array axis index: x is dim 2 */
        if (stages && st == ORACLE_OK) memcpy(stages + (size_t)i * tot, a, sizeof(cplx) * (size_t)tot);
    }
    if (st != ORACLE_OK) { free(a); return st; }

    /* V^F(k) = K^F(k) rho^F(k)   (Eq. 3) */
    for (long long kz = 0; kz < S[2]; ++kz)
        for (long long ky = 0; ky < S[1]; ++ky)
            for (long long kx = 0; kx < S[0]; ++kx) {
                if (Kf_half) {          /* real spectrum: K(-r) = K(r), the other half is K_f(-k) = K_f(k) */
                    double kf;
                    if (kx < H) kf = Kf_half[(kz * S[1] + ky) * H + kx];
                    else        kf = Kf_half[(wrap(-kz, S[2]) * S[1] + wrap(-ky, S[1])) * H + (S[0] - kx)];
                    a[(kz * S[1] + ky) * S[0] + kx] *= kf;
                } else {                /* complex spectrum of a real K: the other half is K_f(-k) = conj K_f(k) */
                    cplx kf;
                    if (kx < H) kf = Kf_half_c[(kz * S[1] + ky) * H + kx];
                    else        kf = conj(Kf_half_c[(wrap(-kz, S[2]) * S[1] + wrap(-ky, S[1])) * H + (S[0] - kx)]);
                    a[(kz * S[1] + ky) * S[0] + kx] *= kf;
                }
            }
    if (stages) memcpy(stages + (size_t)3 * tot, a, sizeof(cplx) * (size_t)tot);

    for (int i = 2; i >= 0 && st == ORACLE_OK; --i) {
        st = oracle_dft_axis(a, dims, 2 - order[i], +1, accum_ld);
        if (stages && st == ORACLE_OK && i > 0)
            memcpy(stages + (size_t)(4 + (2 - i)) * tot, a, sizeof(cplx) * (size_t)tot);
    }
    if (st != ORACLE_OK) { free(a); return st; }

    const double scale = 1.0 / ((double)S[0] * (double)S[1] * (double)S[2]);
    double mi = 0.0;
    for (long long z = 0; z < n[2]; ++z)
        for (long long y = 0; y < n[1]; ++y)
            for (long long x = 0; x < n[0]; ++x) {
                const cplx v = a[(z * S[1] + y) * S[0] + x];
                V[(z * n[1] + y) * n[0] + x] = creal(v) * scale;
                const double im = fabs(cimag(v)) * scale;
                if (im > mi) mi = im;
            }
    if (max_abs_imag_V) *max_abs_imag_V = mi;
    free(a);
    return ORACLE_OK;
}

int oracle_solve(const double *rho, const double *Kf_half, double *V, const long long n[3],
                 const int bc[3], const int axis_order[3], cplx *stages, double *max_abs_imag_V,
                 int accum_ld)
{
    if (!Kf_half) return ORACLE_EINVAL;
    return solve_core(rho, Kf_half, NULL, V, n, bc, axis_order, stages, max_abs_imag_V, accum_ld);
}

/* Eq. 3 with the COMPLEX half spectrum [Sz][Sy][Sx/2+1] of a real kernel without inversion symmetry. */
int oracle_solve_c(const double *rho, const cplx *Kf_half_c, double *V, const long long n[3],
                   const int bc[3], const int axis_order[3], cplx *stages, double *max_abs_imag_V,
                   int accum_ld)
{
    if (!Kf_half_c) return ORACLE_EINVAL;
    return solve_core(rho, NULL, Kf_half_c, V, n, bc, axis_order, stages, max_abs_imag_V, accum_ld);
}

/* ---- Eq. 2 brute force at a list of output points (flat indices into [nz][ny][nx]).
 *  K real-space [Sz][Sy][Sx], origin at index 0, wrap-around order. ---- */
int oracle_direct_sum_at(const double *rho, const double *K, const long long n[3], const int bc[3],
                         const long long *points, long long npoints, double *out)
{
    if (!rho || !K || !n || !bc || !points || !out) return ORACLE_EINVAL;
    long long S[3];
    for (int a = 0; a < 3; ++a) S[a] = n[a] * (bc[a] == 0 ? 2 : 1);
#pragma omp parallel for schedule(dynamic)
    for (long long p = 0; p < npoints; ++p) {
        const long long ix = points[p] % n[0];
        const long long iy = (points[p] / n[0]) % n[1];
        const long long iz = points[p] / (n[0] * n[1]);
        long double acc = 0.0L;
        for (long long z = 0; z < n[2]; ++z) {
            const long long dz = wrap(iz - z, S[2]);
            for (long long y = 0; y < n[1]; ++y) {
                const long long dy = wrap(iy - y, S[1]);
                const double *Krow = K + (dz * S[1] + dy) * S[0];
                const double *rrow = rho + (z * n[1] + y) * n[0];
                long double row = 0.0L;
                for (long long x = 0; x < n[0]; ++x) row += (long double)Krow[wrap(ix - x, S[0])] * rrow[x];
                acc += row;
            }
        }
        out[p] = (double)acc;
    }
    return ORACLE_OK;
}

/* Eq. 2 brute force over the whole box (tiny grids only: O(N^2)). */
int oracle_direct_sum(const double *rho, const double *K, const long long n[3], const int bc[3], double *V)
{
    if (!n) return ORACLE_EINVAL;
    const long long tot = n[0] * n[1] * n[2];
    long long *pts = (long long *)malloc(sizeof(long long) * (size_t)tot);
    if (!pts) return ORACLE_ENOMEM;
    for (long long i = 0; i < tot; ++i) pts[i] = i;
    int st = oracle_direct_sum_at(rho, K, n, bc, pts, tot, V);
    free(pts);
    return st;
}
