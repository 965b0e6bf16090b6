// registry.hpp -- table of compiled pass kernels.  Each inst_*.cu translation unit registers the
// instantiations it holds; api.cu looks kernels up by (kind, S, pruned, lanes_p, precision).
#pragma once

#include <cstddef>
#include <vector>

#include "passes.cuh"   // PassKind

namespace pfft {

struct KernelEntry {
    int kind;      // PassKind
    int S;         // transform length
    int pruned;    // 1: zero-padded axis (spread / compactification fused), 0: periodic axis
    int lanes_p;   // 1: lanes along the pencil index (strided pencils), 0: lanes along the transform
    int prec;      // 0 fp64, 1 fp32
    int variant;   // tuning variant (0 = default; others selectable with POISSON_VARIANT for experiments)
    int nbuf, tws, minb, stg;
    int RA, RB;    // S = RA * RB: radix of the first / second register pass
    int P, TPP, V, NT;
    size_t smem_bytes;
    const void *func;  // __global__ void (*)(PassParams)
    // any-length kernel (generic_pass.cuh): a per-plan entry with run-time length, tile width and radix list
    int generic;       // 0 for the compiled register-engine kernels
    int gen_nfac, gen_fac[16];
    int gen_L, gen_blue;   // transform / buffer length (S, or Bluestein's M) and the Bluestein flag
};

// A fused solve kernel (solve_kernel.cuh): all five passes of one (axis a, axis b, axis c) combination.
struct FusedEntry {
    int prec;
    int S[3], pruned[3], lanes_p[3];   // per processed axis a, b, c
    int P[3];                          // pencils per tile of F1/I1, F2/I2, F3
    int NT, minb;
    size_t smem_bytes;
    const void *func;                  // __global__ void (*)(SolveParams)
};

std::vector<KernelEntry> &kernel_registry();
std::vector<FusedEntry> &fused_registry();
const FusedEntry *find_fused(int prec, const int S[3], const int pruned[3], const int lanes_p[3]);
const KernelEntry *find_kernel(int kind, int S, int pruned, int lanes_p, int prec, int variant = -1);
bool length_supported(int S);

}  // namespace pfft
