/*
 * ia_kernels.cuh -- declarations shared by the translation units of libia_b200.so (host side).
 */
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/ia.h"
#include "ia_dev.cuh"

/* generator description as the device sees it (readings R1-R3) */
struct IaGen {
    int mode, domain, phase_mode;
    unsigned n_theta, n_phi;
    unsigned long long n, first_index, seed;
    unsigned cell;
    const double *y0, *phase;
    double phase0;
    double E_min_uK, log_E_ratio; /* E_uK = E_min exp(u4 log(E_max/E_min)); log_E_ratio = 0 -> fixed */
    double E_fixed_au, v0_fixed;  /* fixed-energy case, computed on the host                        */
    double theta_span_pi, phi_span_pi; /* angular spans in units of pi: 0.5/0.5 octant, 1/2 sphere   */
};

struct IaOut {
    ia_record *records;
    ia_summary *summary;
    double *ic_dump;
};

/* persistent propagation kernel: returns cudaError of the launch */
cudaError_t ia_launch_persistent(const IaParams &P, const IaGen &G, const IaOut &O, unsigned long long *counter,
                                 unsigned long long warn, int grid_blocks, cudaStream_t st);
cudaError_t ia_persistent_info(int device, int *blocks_per_sm, int *threads_per_block, int *regs, int *local_bytes);
cudaError_t ia_launch_generate(const IaParams &P, const IaGen &G, double *ic_dump, cudaStream_t st);

/* verification kernels, two arithmetic variants */
cudaError_t ia_launch_step_map_fma(const IaParams &P, unsigned long long n, const double *t_frac, const double *phase,
                                   const double *y, const double *h, double *ynew, double *err, cudaStream_t st);
cudaError_t ia_launch_step_map_nofma(const IaParams &P, unsigned long long n, const double *t_frac,
                                     const double *phase, const double *y, const double *h, double *ynew,
                                     double *err, cudaStream_t st);
struct IaY12 {
    double y[12];
};
cudaError_t ia_launch_trace_fma(const IaParams &P, IaY12 y0, double phase, double h, unsigned nsteps, double *states,
                                cudaStream_t st);
cudaError_t ia_launch_trace_nofma(const IaParams &P, IaY12 y0, double phase, double h, unsigned nsteps,
                                  double *states, cudaStream_t st);

/* DFMA peak microbenchmark */
cudaError_t ia_run_fp64_peak(int device, double target_ms, double *tflops, double *elapsed_ms);
