/*
 * ia_nofma.cu -- the verification kernels built WITHOUT floating-point contraction
 * (nvcc -fmad=false; BASELINE.json north_star: "a fixed-step mode built with fmad off").
 * Same source as the production arithmetic (ia_dev.cuh); only the explicit fma() calls of the
 * reciprocal refinement, fifth root and cosine range reduction remain fused.
 */
#include "ia_kernels.cuh"

#define IA_VARIANT nofma
#include "ia_verify.cuh"
