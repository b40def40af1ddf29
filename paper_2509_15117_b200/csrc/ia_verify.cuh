/*
 * ia_verify.cuh -- verification kernels (K3), textually included once per arithmetic variant:
 * ia_kernels.cu defines IA_VARIANT = fma (production arithmetic), ia_nofma.cu defines
 * IA_VARIANT = nofma and is compiled with -fmad=false (BASELINE.json north_star: "fixed-step mode
 * built with fmad off").  Both call the same ia_dp5_attempt as the persistent kernel.
 */
#ifndef IA_VARIANT
#error "define IA_VARIANT before including ia_verify.cuh"
#endif
#define IA_CAT2(a, b) a##b
#define IA_CAT(a, b) IA_CAT2(a, b)
#define IA_NAME(base) IA_CAT(base, IA_VARIANT)

/* n independent uncontrolled steps: the one-step map of reading R12(i) */
__global__ void IA_NAME(ia_step_map_kernel_)(const __grid_constant__ IaParams P, unsigned long long n,
                                             const double *t_frac, const double *phase, const double *y,
                                             const double *h, double *ynew, double *err_out) {
    const unsigned long long j = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    double x[6], v[6], A1[6], xn[6], vn[6], A7[6], r2, s, r2n;
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        x[i] = y[j * 12 + i];
        v[i] = y[j * 12 + 6 + i];
    }
    const double tf = t_frac[j], ph = phase[j];
    ia_accel(P, x, ia_cos_folded(P.omega * tf + ph), A1, r2, s);
    IaErr err;
    bool finite;
    ia_dp5_attempt(P, x, v, A1, tf, ph, h[j], xn, vn, A7, r2n, err, finite);
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        ynew[j * 12 + i] = xn[i];
        ynew[j * 12 + 6 + i] = vn[i];
    }
    if (err_out != nullptr) err_out[j] = finite ? err.num / err.den : __longlong_as_double(0x7ff8000000000000ll);
}

/* nsteps uncontrolled steps of one trajectory, every state written out (reading R12(ii)) */
__global__ void IA_NAME(ia_trace_kernel_)(const __grid_constant__ IaParams P, IaY12 y0, double phase, double h,
                                          unsigned nsteps, double *states) {
    if (blockIdx.x != 0 || threadIdx.x != 0) return;
    double x[6], v[6], A1[6], xn[6], vn[6], A7[6], r2, s, r2n;
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        x[i] = y0.y[i];
        v[i] = y0.y[6 + i];
    }
    double tf = 0.0;
    unsigned n_per = 0;
    states[0] = 0.0;
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        states[1 + i] = x[i];
        states[7 + i] = v[i];
    }
    ia_accel(P, x, ia_cos_folded(phase), A1, r2, s);
    for (unsigned n = 0; n < nsteps; ++n) {
        IaErr err;
        bool finite;
        ia_dp5_attempt(P, x, v, A1, tf, phase, h, xn, vn, A7, r2n, err, finite);
        tf += h;
        if (tf >= P.T_rf) {
            tf -= P.T_rf;
            ++n_per;
        }
#pragma unroll
        for (int i = 0; i < 6; ++i) {
            x[i] = xn[i];
            v[i] = vn[i];
            A1[i] = A7[i];
        }
        double *o = states + (unsigned long long)(n + 1) * 13;
        o[0] = (double)n_per * P.T_rf + tf;
#pragma unroll
        for (int i = 0; i < 6; ++i) {
            o[1 + i] = x[i];
            o[7 + i] = v[i];
        }
    }
}

cudaError_t IA_NAME(ia_launch_step_map_)(const IaParams &P, unsigned long long n, const double *t_frac,
                                         const double *phase, const double *y, const double *h, double *ynew,
                                         double *err, cudaStream_t st) {
    if (n == 0) return cudaSuccess;
    const unsigned threads = 64;
    IA_NAME(ia_step_map_kernel_)<<<(unsigned)((n + threads - 1) / threads), threads, 0, st>>>(P, n, t_frac, phase, y,
                                                                                              h, ynew, err);
    return cudaGetLastError();
}

cudaError_t IA_NAME(ia_launch_trace_)(const IaParams &P, IaY12 y0, double phase, double h, unsigned nsteps,
                                      double *states, cudaStream_t st) {
    IA_NAME(ia_trace_kernel_)<<<1, 32, 0, st>>>(P, y0, phase, h, nsteps, states);
    return cudaGetLastError();
}
