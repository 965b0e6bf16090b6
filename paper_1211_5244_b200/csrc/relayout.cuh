// relayout.cuh -- where each slot of the internal K^F copy comes from ("a transposition
// of the associated kernel ... carried out only once").
// Internal order: kint[((tile*(V/KVEC) + q)*NT + tid)*KVEC + j], r = q*KVEC + j, KVEC = 16 bytes of
// reals -- exactly the 16-byte vectors thread `tid` of pass F3 consumes for its registers r, so the
// multiply of Eq. 3 streams K^F with perfectly coalesced 128-bit accesses and no index arithmetic.
#pragma once

#include "fft_core.cuh"

namespace pfft {

struct RelayoutParams {
    int RA, RB, TPP, P, V, NT, lanes_p;
    int tiles_per_g, n_p;
    int fold;             // 0, or S_b: only pencils 0 .. S_b / 2 are stored (K^F even along axis b, poisson_set_kernel_even)
    int g0;               // first k_a plane held (sharded plans keep only their own planes; else 0)
    int a_axis, c_axis;   // the pencil index pp runs along the remaining axis
    int sx, sy, sz;
    long long total;
    double scale;  // 1/(S_x S_y S_z)
};

template <typename T>
PF_HD T relayout_value(const T *kuser, const RelayoutParams &q, long long idx) {
    const int kvec = 16 / (int)sizeof(T);
    const int tid = (int)((idx / kvec) % q.NT);
    const int r = (int)((idx / ((long long)kvec * q.NT)) % (q.V / kvec)) * kvec + (int)(idx % kvec);
    const long long tile = idx / ((long long)q.NT * q.V);
    int t, p;
    if (q.lanes_p) { p = tid % q.P; t = tid / q.P; } else { t = tid % q.TPP; p = tid / q.TPP; }
    const long long g = tile / q.tiles_per_g + q.g0;
    const long long pp = (tile % q.tiles_per_g) * q.P + p;
    if (pp >= q.n_p || (q.fold && pp > q.fold / 2)) return (T)0;   // folded storage keeps pencils 0 .. S_b / 2 (q.tiles_per_g tiles of them)
    const int i = r / q.RB, k1 = r % q.RB;
    if (t + q.TPP * i >= q.RA) return (T)0;      // ragged last column of layout B: this thread owns no k2 there
    const int kc = (t + q.TPP * i) + q.RA * k1;  // layout B of passes.cuh: k = k2 + RA*k1
    long long f[3];
    f[3 - q.a_axis - q.c_axis] = pp; f[q.c_axis] = kc; f[q.a_axis] = g;
    long long kx = f[0], ky = f[1], kz = f[2];
    const int hx = q.sx / 2 + 1;
    if (kx > q.sx / 2) {  // K^F(-k) = K^F(k): the half the caller did not pass
        kx = q.sx - kx; ky = (q.sy - ky) % q.sy; kz = (q.sz - kz) % q.sz;
    }
    return (T)((double)kuser[(kz * q.sy + ky) * hx + kx] * q.scale);
}

}  // namespace pfft
