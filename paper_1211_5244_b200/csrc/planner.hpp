// planner.hpp -- host-only planning for the customised 3D FFT (no CUDA calls; usable without a GPU).
// Decides the axis order (periodic axes first, free axes last), the array extents
// after each pass (an axis is padded only when it is transformed, and dropped back
// to N right after its inverse), and the (g, n, p) addressing of every pass.
#pragma once

#include <cstring>

#include "../../include/poisson.h"

namespace pfft {

struct PassDesc {
    int kind;      // POISSON_PASS_*
    int axis;      // 0 x, 1 y, 2 z
    int S;         // transform length
    int pruned;    // axis is zero padded
    int lanes_p;   // lanes along the pencil index (strided pencils)
    int generic;   // 1: no register-engine kernel covers this pass (length not in sizes.def, or odd N_x in the R2C / C2R
                   //    pass): it runs the any-length kernel of generic_pass.cuh
    int n_real;    // F1 / I1: real pencils along x (= N_x); the generic kernel pairs them (2q, 2q + 1), the last one alone if odd
    long long n_g, n_p;
    long long gs_in, ns_in, ps_in, gs_out, ns_out, ps_out;
};

struct PlanDesc {
    int n[3], bc[3], s[3], prec;
    int order[3];        // a, b, c
    int H;               // S_a/2 + 1
    long long ext1[3];   // A1 extents per axis id (x,y,z): a -> H
    long long ext2[3];   // A2 extents per axis id: a -> H, b -> S_b
    long long a1_elems, a2_elems, kuser_elems;
    PassDesc pass[5];
    poisson_plan_info info;
};

#define PF_GENERIC_MAX_S 4096   // longest transform of the any-length kernel (generic_pass.cuh: GEN_MAX_S)

inline bool length_in_list(int S) {
#define PF_SIZE(S, RA, RB, TPP) S,
    static const int ok[] = {
#include "sizes.def"
    };
#undef PF_SIZE
    for (int v : ok) if (v == S) return true;
    return false;
}

inline int plan_build(int nx, int ny, int nz, const int bc_in[3], int prec, PlanDesc &d) {
    if (!bc_in) return POISSON_EINVAL;
    if (nx <= 0 || ny <= 0 || nz <= 0) return POISSON_EINVAL;
    if (prec != POISSON_FP64 && prec != POISSON_FP32) return POISSON_EINVAL;
    std::memset(&d, 0, sizeof(d));
    d.n[0] = nx; d.n[1] = ny; d.n[2] = nz; d.prec = prec;
    for (int a = 0; a < 3; ++a) {
        if (bc_in[a] != POISSON_BC_FREE && bc_in[a] != POISSON_BC_PERIODIC) return POISSON_EINVAL;
        d.bc[a] = bc_in[a];
        if (d.n[a] > (1 << 20)) return POISSON_EUNSUPPORTED;
        d.s[a] = d.n[a] * (d.bc[a] == POISSON_BC_FREE ? 2 : 1);   // S_i = N_i * B_i
    }
    for (int a = 0; a < 3; ++a)
        if (d.s[a] > PF_GENERIC_MAX_S) return POISSON_EUNSUPPORTED;   // the only refusal: above the any-length kernel's limit
    auto per = [&](int a) { return d.bc[a] == POISSON_BC_PERIODIC; };
    // a: never x (the half spectrum H = S_a/2+1 is odd and would break 128-byte rows on the
    // contiguous axis); periodic preferred, z preferred on a tie.
    int a = per(2) ? 2 : (per(1) ? 1 : 2);
    int o = (a == 2) ? 1 : 2;  // the other non-x axis
    int b, c;
    if (per(0) != per(o)) { b = per(0) ? 0 : o; c = per(0) ? o : 0; }
    else { b = o; c = 0; }       // contiguous axis last: pass F3 streams whole rows
    d.order[0] = a; d.order[1] = b; d.order[2] = c;
    d.H = d.s[a] / 2 + 1;

    for (int q = 0; q < 3; ++q) { d.ext1[q] = d.n[q]; d.ext2[q] = d.n[q]; }
    d.ext1[a] = d.H; d.ext2[a] = d.H; d.ext2[b] = d.s[b];
    d.a1_elems = d.ext1[0] * d.ext1[1] * d.ext1[2];
    d.a2_elems = d.ext2[0] * d.ext2[1] * d.ext2[2];
    d.kuser_elems = (long long)d.s[2] * d.s[1] * (d.s[0] / 2 + 1);

    auto stride = [](const long long ext[3], int q) -> long long {
        return q == 0 ? 1 : (q == 1 ? ext[0] : ext[0] * ext[1]);
    };
    const long long extp[3] = {d.n[0] / 2, d.n[1], d.n[2]};  // rho / V read as x-pairs

    // F1 / I1: axis a, strided, pairs along x
    PassDesc f1{}; f1.kind = POISSON_PASS_F1; f1.axis = a; f1.S = d.s[a]; f1.pruned = !per(a); f1.lanes_p = 1;
    f1.generic = !length_in_list(d.s[a]) || d.n[0] % 2 != 0;
    f1.n_real = d.n[0];
    f1.n_g = d.n[o];
    if (!f1.generic) {   // register engine: rho / V read as x-pairs (one 16-byte access per pair)
        f1.n_p = d.n[0] / 2;
        f1.gs_in = stride(extp, o); f1.ns_in = stride(extp, a); f1.ps_in = 1;
    } else {             // any-length kernel: strides in REAL elements, ceil(N_x / 2) pair pencils
        const long long extr[3] = {d.n[0], d.n[1], d.n[2]};
        f1.n_p = (d.n[0] + 1) / 2;
        f1.gs_in = stride(extr, o); f1.ns_in = stride(extr, a); f1.ps_in = 1;
    }
    f1.gs_out = stride(d.ext1, o); f1.ns_out = stride(d.ext1, a); f1.ps_out = 1;
    PassDesc i1 = f1; i1.kind = POISSON_PASS_I1;
    i1.gs_in = f1.gs_out; i1.ns_in = f1.ns_out; i1.ps_in = f1.ps_out;
    i1.gs_out = f1.gs_in; i1.ns_out = f1.ns_in; i1.ps_out = f1.ps_in;

    // F2 / I2: axis b
    PassDesc f2{}; f2.kind = POISSON_PASS_F2; f2.axis = b; f2.S = d.s[b]; f2.pruned = !per(b);
    f2.generic = !length_in_list(d.s[b]);
    // every middle pass works plane by plane: g = k_a (n_g = H), so that F3 / I2 of a plane depend on that plane only
    if (b == 0) {   // contiguous pencils along x, one per point of the remaining axis c
        f2.lanes_p = 0; f2.n_g = d.H; f2.n_p = d.ext1[c];
        f2.gs_in = stride(d.ext1, a); f2.ns_in = 1; f2.ps_in = stride(d.ext1, c);
        f2.gs_out = stride(d.ext2, a); f2.ns_out = 1; f2.ps_out = stride(d.ext2, c);
    } else {
        f2.lanes_p = 1; f2.n_g = d.H; f2.n_p = d.ext1[0];
        f2.gs_in = stride(d.ext1, a); f2.ns_in = stride(d.ext1, b); f2.ps_in = 1;
        f2.gs_out = stride(d.ext2, a); f2.ns_out = stride(d.ext2, b); f2.ps_out = 1;
    }
    PassDesc i2 = f2; i2.kind = POISSON_PASS_I2;
    i2.gs_in = f2.gs_out; i2.ns_in = f2.ns_out; i2.ps_in = f2.ps_out;
    i2.gs_out = f2.gs_in; i2.ns_out = f2.ns_in; i2.ps_out = f2.ps_in;

    // F3: axis c, in place on A2
    PassDesc f3{}; f3.kind = POISSON_PASS_F3; f3.axis = c; f3.S = d.s[c]; f3.pruned = !per(c);
    f3.generic = !length_in_list(d.s[c]);
    if (c == 0) {   // contiguous pencils along x, one per point of axis b (already at its padded length S_b)
        f3.lanes_p = 0; f3.n_g = d.H; f3.n_p = d.ext2[b];
        f3.gs_in = stride(d.ext2, a); f3.ns_in = 1; f3.ps_in = stride(d.ext2, b);
    } else {
        f3.lanes_p = 1; f3.n_g = d.H; f3.n_p = d.ext2[0];
        f3.gs_in = stride(d.ext2, a); f3.ns_in = stride(d.ext2, c); f3.ps_in = 1;
    }
    f3.gs_out = f3.gs_in; f3.ns_out = f3.ns_in; f3.ps_out = f3.ps_in;

    d.pass[0] = f1; d.pass[1] = f2; d.pass[2] = f3; d.pass[3] = i2; d.pass[4] = i1;

    // ---- host-side description (include/poisson.h)
    poisson_plan_info &I = d.info;
    const long long r = prec == POISSON_FP64 ? 8 : 4;
    for (int q = 0; q < 3; ++q) { I.n[q] = d.n[q]; I.bc[q] = d.bc[q]; I.s[q] = d.s[q]; I.order[q] = d.order[q]; }
    I.precision = prec; I.half_len = d.H;
    const long long rho_b = (long long)nx * ny * nz * r;
    const long long a1_b = d.a1_elems * 2 * r, a2_b = d.a2_elems * 2 * r;
    const long long k_b = (long long)d.H * d.s[b] * d.s[c] * r;
    I.rows[0] = I.rows[4] = (long long)d.n[b] * d.n[c];       // real rows of length S_a
    I.rows[1] = I.rows[3] = (long long)d.H * d.n[c];
    I.rows[2] = (long long)d.H * d.s[b];
    I.length[0] = I.length[4] = d.s[a]; I.length[1] = I.length[3] = d.s[b]; I.length[2] = d.s[c];
    I.bytes[0] = I.bytes[4] = rho_b + a1_b;
    I.bytes[1] = I.bytes[3] = a1_b + a2_b;
    I.bytes[2] = 2 * a2_b + k_b;
    I.bytes_total = 0;
    for (int q = 0; q < 5; ++q) I.bytes_total += I.bytes[q];
    // N_b N_c rows of S_a, then S_a N_c rows of S_b, then S_a S_b rows of S_c,
    // against 3 S_a S_b S_c for the unpruned transform.
    const double sa = d.s[a], sb = d.s[b], sc = d.s[c];
    I.fft_fraction = ((double)d.n[b] * d.n[c] * sa + sa * d.n[c] * sb + sa * sb * sc) / (3.0 * sa * sb * sc);
    I.workspace_bytes = 0;  // filled by poisson_plan_create (depends on tile sizes)
    return POISSON_OK;
}

// ---- sharded single solve ("transposes on the reduced data set", PAPER.md:89 GPU-to-GPU transfers)
// rho / V are distributed along the axis o (the non-x axis that is not a); between F1 and F2, and between I2 and I1, the
// half spectrum A1 changes hands once: distributed along o <-> distributed along k_a.  Both partitions are balanced:
// rank s owns [floor(T s / R), floor(T (s + 1) / R)) of T points, and v belongs to rank floor(((v + 1) R - 1) / T).
inline int shard_lo(int total, int s, int R) { return (int)((long long)total * s / R); }
inline int shard_owner(int total, int v, int R) { return (int)((((long long)v + 1) * R - 1) / total); }

struct ShardDesc {
    int rank, R;
    int a, o;                 // plane axis, split axis
    int o0, o1, k0, k1;       // this rank's slab of rho / V along o, and its planes k_a
    long long ext_rho[3];     // local rho / V extents per axis id (o -> o1 - o0)
    long long ext_mid[3];     // this rank's exchange slab 1: A1 with a -> k1 - k0 (o whole)
    long long ext_a2[3];      // its A2: a -> k1 - k0, b -> S_b
    long long ext_back[3];    // its exchange slab 2: A1 with o -> o1 - o0 (a whole: H)
    long long mid_elems, back_elems, a2_elems;
    PassDesc pass[5];         // F1S (in strides only), F2, F3, I2S (in strides only), I1 on the local arrays
};

inline int shard_build(const PlanDesc &d, int rank, int R, ShardDesc &sh) {
    if (R < 1 || rank < 0 || rank >= R) return POISSON_EINVAL;
    std::memset(&sh, 0, sizeof(sh));
    const int a = d.order[0], b = d.order[1], c = d.order[2], o = 3 - a;
    if (R > d.n[o] || R > d.H || R > 32) return POISSON_EUNSUPPORTED;    // every rank holds a non-empty slab and plane range
    if (d.n[0] % 2 != 0) return POISSON_EUNSUPPORTED;                     // the register-engine R2C pass reads x-pairs
    for (int q = 0; q < 5; ++q) if (d.pass[q].generic) return POISSON_EUNSUPPORTED;
    sh.rank = rank; sh.R = R; sh.a = a; sh.o = o;
    sh.o0 = shard_lo(d.n[o], rank, R); sh.o1 = shard_lo(d.n[o], rank + 1, R);
    sh.k0 = shard_lo(d.H, rank, R);    sh.k1 = shard_lo(d.H, rank + 1, R);
    const long long no = sh.o1 - sh.o0, ng = sh.k1 - sh.k0;
    for (int q = 0; q < 3; ++q) { sh.ext_rho[q] = d.n[q]; sh.ext_mid[q] = d.ext1[q]; sh.ext_a2[q] = d.ext2[q]; sh.ext_back[q] = d.ext1[q]; }
    sh.ext_rho[o] = no; sh.ext_mid[a] = ng; sh.ext_a2[a] = ng; sh.ext_back[o] = no;
    sh.mid_elems = sh.ext_mid[0] * sh.ext_mid[1] * sh.ext_mid[2];
    sh.back_elems = sh.ext_back[0] * sh.ext_back[1] * sh.ext_back[2];
    sh.a2_elems = sh.ext_a2[0] * sh.ext_a2[1] * sh.ext_a2[2];
    auto stride = [](const long long ext[3], int q) -> long long { return q == 0 ? 1 : (q == 1 ? ext[0] : ext[0] * ext[1]); };
    const long long extp[3] = {sh.ext_rho[0] / 2, sh.ext_rho[1], sh.ext_rho[2]};   // rho / V read as x-pairs

    PassDesc f1 = d.pass[0];   // kind, axis, S, pruned, lanes_p as in the global plan
    f1.n_g = no; f1.n_p = d.n[0] / 2;
    f1.gs_in = stride(extp, o); f1.ns_in = stride(extp, a); f1.ps_in = 1;
    f1.gs_out = f1.ns_out = f1.ps_out = 0;                                        // scattered over the ranks' slabs (PassParams::sh_*)
    PassDesc i1 = d.pass[4];
    i1.n_g = no; i1.n_p = d.n[0] / 2;
    i1.gs_in = stride(sh.ext_back, o); i1.ns_in = stride(sh.ext_back, a); i1.ps_in = 1;
    i1.gs_out = f1.gs_in; i1.ns_out = f1.ns_in; i1.ps_out = 1;

    PassDesc f2 = d.pass[1];
    f2.n_g = ng;
    if (b == 0) { f2.n_p = sh.ext_mid[c];
        f2.gs_in = stride(sh.ext_mid, a); f2.ns_in = 1; f2.ps_in = stride(sh.ext_mid, c);
        f2.gs_out = stride(sh.ext_a2, a); f2.ns_out = 1; f2.ps_out = stride(sh.ext_a2, c);
    } else { f2.n_p = sh.ext_mid[0];
        f2.gs_in = stride(sh.ext_mid, a); f2.ns_in = stride(sh.ext_mid, b); f2.ps_in = 1;
        f2.gs_out = stride(sh.ext_a2, a); f2.ns_out = stride(sh.ext_a2, b); f2.ps_out = 1;
    }
    PassDesc i2 = d.pass[3];
    i2.n_g = ng; i2.n_p = f2.n_p;
    i2.gs_in = f2.gs_out; i2.ns_in = f2.ns_out; i2.ps_in = f2.ps_out;
    i2.gs_out = i2.ns_out = i2.ps_out = 0;                                        // scattered
    PassDesc f3 = d.pass[2];
    f3.n_g = ng;
    if (c == 0) { f3.n_p = sh.ext_a2[b]; f3.gs_in = stride(sh.ext_a2, a); f3.ns_in = 1; f3.ps_in = stride(sh.ext_a2, b); }
    else { f3.n_p = sh.ext_a2[0]; f3.gs_in = stride(sh.ext_a2, a); f3.ns_in = stride(sh.ext_a2, c); f3.ps_in = 1; }
    f3.gs_out = f3.gs_in; f3.ns_out = f3.ns_in; f3.ps_out = f3.ps_in;
    sh.pass[0] = f1; sh.pass[1] = f2; sh.pass[2] = f3; sh.pass[3] = i2; sh.pass[4] = i1;
    return POISSON_OK;
}

}  // namespace pfft
