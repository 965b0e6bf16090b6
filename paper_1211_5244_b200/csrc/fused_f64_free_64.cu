// Fused solve kernels (solve_kernel.cuh): PF_FUSED(T, prec, SA, PA, SB, PB, LB, SC, PC, LC, MINB), see fused_inst.cuh.
#define PF_FUSED_LIST PF_FUSED(double,0,64,1,64,1,1,64,1,0,0)
#include "fused_inst.cuh"
