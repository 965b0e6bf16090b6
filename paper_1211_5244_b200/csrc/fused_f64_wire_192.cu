// Fused solve kernels (solve_kernel.cuh): PF_FUSED(T, prec, SA, PA, SB, PB, LB, SC, PC, LC, MINB), see fused_inst.cuh.
#define PF_FUSED_LIST PF_FUSED(double,0,256,0,192,1,1,192,1,0,0)
#include "fused_inst.cuh"
