// Fused solve kernels (solve_kernel.cuh): PF_FUSED(T, prec, SA, PA, SB, PB, LB, SC, PC, LC, MINB), see fused_inst.cuh.
#define PF_FUSED_LIST PF_FUSED(double,0,8,1,8,1,1,8,1,0,0) PF_FUSED(double,0,16,1,16,1,1,16,1,0,0) PF_FUSED(double,0,32,1,32,1,1,32,1,0,0) PF_FUSED(double,0,16,0,16,0,1,16,0,0,0) PF_FUSED(double,0,24,1,48,1,1,12,1,0,0)
#include "fused_inst.cuh"
