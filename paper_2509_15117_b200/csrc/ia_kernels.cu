/*
 * ia_kernels.cu -- the persistent propagation kernel (K1), the initial-condition generator (K2)
 * and the production-arithmetic build of the verification kernels (K3).
 *
 * K1: one lane = one trajectory.  State, accelerations of all seven stages, step size and event
 * bookkeeping live in registers; nothing per step touches memory.  A lane whose trajectory has
 * terminated writes its 64-byte record, adds to the ensemble summary and takes the next index from
 * a global work counter (one atomicAdd per warp-refill), so warps stay full although trajectory
 * lengths span 10^3..10^7 steps.
 * Exit localisation (reading R7) re-uses the same step body with the lane in mode LOC, so the warp
 * never diverges on it.
 */
#include "ia_kernels.cuh"

#define IA_WARPS_PER_BLOCK 1
#define IA_THREADS (32 * IA_WARPS_PER_BLOCK)
#define IA_FULL 0xffffffffu

enum { MODE_IDLE = 0, MODE_RUN = 1, MODE_LOC = 2 };

/* ---- generator (readings R1-R3) ------------------------------------------------------------ */

/* Philox4x32-10 (Salmon et al., SC'11), from the published round function. */
__device__ __forceinline__ void ia_philox(unsigned c0, unsigned c1, unsigned c2, unsigned c3, unsigned k0, unsigned k1,
                                          unsigned (&out)[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned lo0 = 0xD2511F53u * c0, hi0 = __umulhi(0xD2511F53u, c0);
        const unsigned lo1 = 0xCD9E8D57u * c2, hi1 = __umulhi(0xCD9E8D57u, c2);
        const unsigned n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* 53-bit uniform in (0,1) from two words (reading R2) */
__device__ __forceinline__ double ia_u53(unsigned we, unsigned wo) {
    return ((double)(we >> 5) * 67108864.0 + (double)(wo >> 6) + 0.5) * (1.0 / 9007199254740992.0);
}

/* Initial condition of local trajectory j: x = (r_i, r_a), v = (v_i, v_a), rf phase, energy. */
__device__ __noinline__ void ia_generate_ic(const IaParams &P, const IaGen &G, unsigned long long j, double (&x)[6],
                                            double (&v)[6], double &phase, double &E_au) {
    if (G.mode == IA_IC_EXPLICIT) {
#pragma unroll
        for (int i = 0; i < 6; ++i) {
            x[i] = G.y0[j * 12 + i];
            v[i] = G.y0[j * 12 + 6 + i];
        }
        phase = G.phase[j];
        E_au = 0.5 * P.m_a * (v[3] * v[3] + v[4] * v[4] + v[5] * v[5]);
        return;
    }
    const unsigned long long gi = G.first_index + j;
    unsigned w0[4], w1[4];
    ia_philox((unsigned)gi, (unsigned)(gi >> 32), G.cell, 0u, (unsigned)G.seed, (unsigned)(G.seed >> 32), w0);
    ia_philox((unsigned)gi, (unsigned)(gi >> 32), G.cell, 1u, (unsigned)G.seed, (unsigned)(G.seed >> 32), w1);
    const double u1 = ia_u53(w0[0], w0[1]), u2 = ia_u53(w0[2], w0[3]);
    const double u3 = ia_u53(w1[0], w1[1]), u4 = ia_u53(w1[2], w1[3]);
    double ct, st, sp, cp;
    if (G.mode == IA_IC_GRID) {
        const unsigned long long ii = gi / G.n_phi, jj = gi % G.n_phi;
        /* theta = (i + 1/2) span / n_theta, evaluated as sincospi(theta/pi) */
        sincospi(((double)ii + 0.5) * G.theta_span_pi / (double)G.n_theta, &st, &ct);
        sincospi(((double)jj + 0.5) * G.phi_span_pi / (double)G.n_phi, &sp, &cp);
    } else {
        ct = (G.domain == 0) ? u1 : 2.0 * u1 - 1.0;
        st = sqrt(1.0 - ct * ct);
        sincospi(G.phi_span_pi * u2, &sp, &cp);
    }
    phase = (G.phase_mode == 1) ? 6.28318530717958647692 * u3 : G.phase0;
    double v0;
    if (G.log_E_ratio != 0.0) {
        const double E_uK = G.E_min_uK * exp(u4 * G.log_E_ratio);
        E_au = E_uK * 1e-6 * 3.1668115634564e-6; /* k_B in E_h/K (CODATA 2022) */
        v0 = sqrt(2.0 * E_au / P.m_a);
    } else {
        E_au = G.E_fixed_au;
        v0 = G.v0_fixed;
    }
    const double n0 = st * cp, n1 = st * sp, n2 = ct;
    x[0] = 0.0; x[1] = 0.0; x[2] = 0.0;           /* ion at the trap centre, at rest */
    v[0] = 0.0; v[1] = 0.0; v[2] = 0.0;
    x[3] = P.r0 * n0; x[4] = P.r0 * n1; x[5] = P.r0 * n2;   /* atom on the r0 sphere ...            */
    v[3] = -v0 * n0; v[4] = -v0 * n1; v[5] = -v0 * n2;      /* ... aimed at the ion                */
}

__global__ void ia_generate_kernel(IaParams P, IaGen G, double *ic_dump) {
    const unsigned long long j = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= G.n) return;
    double x[6], v[6], phase, E;
    ia_generate_ic(P, G, j, x, v, phase, E);
    double *o = ic_dump + j * 14;
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        o[i] = x[i];
        o[6 + i] = v[i];
    }
    o[12] = phase;
    o[13] = E;
}

/* ---- per-trajectory set-up (reading R5: ode45 initial step) --------------------------------- */

__device__ __forceinline__ bool ia_isfinite(double a) { return fabs(a) <= 1.79769313486231570815e308; }

__device__ __forceinline__ unsigned long long ia_globaltimer() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}

/* ---- K1 ------------------------------------------------------------------------------------- */

__global__ void __launch_bounds__(IA_THREADS) ia_persistent_kernel(const __grid_constant__ IaParams P,
                                                                  const __grid_constant__ IaGen G, IaOut O,
                                                                  unsigned long long *counter,
                                                                  unsigned long long warn) {
    const unsigned lane = threadIdx.x & 31u;
    /* lane state */
    double x[6], v[6], A1[6];
    double tf = 0.0, h = 0.0, phase = 0.0, s_old = 0.0, t_first = 0.0, t_last = 0.0;
    unsigned n_per = 0, n_coll = 0, n_tp = 0, steps_acc = 0, steps_rej = 0, n_loc = 0;
    unsigned long long slot = 0;
    int mode = MODE_IDLE;
    bool failed = false, exhausted = false;
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        x[i] = (i < 3) ? 0.0 : 1.0 + i; /* harmless finite state for idle lanes */
        v[i] = 0.0;
        A1[i] = 0.0;
    }
    if (O.summary != nullptr && threadIdx.x == 0) {
        const unsigned long long t0 = ia_globaltimer();
        if (blockIdx.x == 0) {
            atomicCAS((unsigned long long *)&O.summary->t_start_ns, 0ull, t0);
            if (warn) atomicOr((unsigned long long *)&O.summary->warn, warn);
        }
    }

    for (;;) {
        /* ---- refill idle lanes from the global work counter (a12) ---- */
        const bool want = (mode == MODE_IDLE) && !exhausted;
        const unsigned wm = __ballot_sync(IA_FULL, want);
        if (wm) {
            const int leader = __ffs(wm) - 1;
            unsigned long long base = 0;
            if ((int)lane == leader) base = atomicAdd(counter, (unsigned long long)__popc(wm));
            base = __shfl_sync(IA_FULL, base, leader);
            if (want) {
                const unsigned long long j = base + __popc(wm & ((1u << lane) - 1u));
                if (j >= G.n) {
                    exhausted = true;
                    if (O.summary != nullptr)
                        atomicCAS((unsigned long long *)&O.summary->t_first_idle_ns, 0ull, ia_globaltimer());
                } else {
                    double E_au;
                    ia_generate_ic(P, G, j, x, v, phase, E_au);
                    if (O.ic_dump != nullptr) {
                        double *o = O.ic_dump + j * 14;
#pragma unroll
                        for (int i = 0; i < 6; ++i) {
                            o[i] = x[i];
                            o[6 + i] = v[i];
                        }
                        o[12] = phase;
                        o[13] = E_au;
                    }
                    slot = j;
                    tf = 0.0; n_per = 0; n_coll = 0; n_tp = 0; steps_acc = 0; steps_rej = 0; n_loc = 0;
                    t_first = 0.0; t_last = 0.0; failed = false;
                    bool ok = ia_isfinite(phase);
#pragma unroll
                    for (int i = 0; i < 6; ++i) ok = ok && ia_isfinite(x[i]) && ia_isfinite(v[i]);
                    if (!ok) {
                        /* status 3: non-finite initial state; record it and stay idle */
                        if (O.records != nullptr) {
                            ia_record r;
                            r.ke_ion = 0.5 * P.m_i * (v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
                            r.t_dwell = 0.0; r.t_life = 0.0;
                            r.va_f[0] = v[3]; r.va_f[1] = v[4]; r.va_f[2] = v[5];
                            r.n_coll = 0; r.n_tp = 0; r.steps_acc = 0; r.steps_rej = 0; r.status = 3; r.n_loc = 0;
                            O.records[j] = r;
                        }
                        if (O.summary != nullptr) {
                            atomicAdd((unsigned long long *)&O.summary->n_done, 1ull);
                            atomicAdd((unsigned long long *)&O.summary->n_status[3], 1ull);
                            atomicAdd((unsigned long long *)&O.summary->hist_ncoll[0], 1ull);
                        }
#pragma unroll
                        for (int i = 0; i < 6; ++i) {
                            x[i] = (i < 3) ? 0.0 : 1.0 + i;
                            v[i] = 0.0;
                        }
                        phase = 0.0;
                    } else {
                        /* keep the cosine argument in the folded range for any caller-supplied phase */
                        if (fabs(phase) > 6.5) phase -= 6.28318530717958647692 * rint(phase * 0.15915494309189533577);
                        double r2, s;
                        ia_accel(P, x, ia_cos_folded(phase), A1, r2, s);
                        /* h = min(h_max, t_max); rho = ||f0 / max(|y0|, thr)||_inf / (0.8 rtol^(1/5)) */
                        double rho = 0.0;
#pragma unroll
                        for (int i = 0; i < 6; ++i) {
                            rho = fmax(rho, fabs(v[i]) / fmax(fabs(x[i]), P.thr));
                            rho = fmax(rho, fabs(A1[i]) / fmax(fabs(v[i]), P.thr));
                        }
                        rho = rho / P.h0_scale;
                        h = fmin(P.h_max, P.t_max);
                        if (h * rho > 1.0) h = 1.0 / rho;
                        if (h < P.h_min) h = P.h_min;
                        s_old = ia_sdot(x, v);
                        mode = MODE_RUN;
                    }
                }
            }
        }
        if (!__any_sync(IA_FULL, mode != MODE_IDLE)) {
            if (__all_sync(IA_FULL, exhausted)) break;
            continue;
        }

        /* ---- one DP5(4) attempt for every lane (idle lanes step a harmless dummy state) ---- */
        bool last = false;
        if (mode == MODE_RUN) {
            /* clip the last step to land on t_max (R5/R8) */
            const double rem = (P.t_max_rf - (double)n_per) * P.T_rf - tf;
            if (h >= rem) {
                h = rem;
                last = true;
            }
        }
        double xn[6], vn[6], A7[6], r2n;
        IaErr err;
        bool finite;
        ia_dp5_attempt(P, x, v, A1, tf, phase, h, xn, vn, A7, r2n, err, finite);

        if (mode != MODE_IDLE) {
            /* controller quantities, common to accept and reject: yq = (rtol/err)^(1/5) */
            const bool accept = finite && (err.num <= P.rtol * err.den);
            double xr = err.num * ia_rcp(err.den * P.rtol);
            if (!finite) xr = 1e30;
            xr = fmax(fmin(xr, 1e30), 1e-30); /* NaN -> 1e30 (fmin returns the non-NaN operand) */
            const double yq = ia_inv_fifth_root(xr);
            const double s_new = ia_sdot(xn, vn);
            const double now = (double)n_per * P.T_rf + tf;
            int fin = -1;          /* >= 0: terminate with this status */
            bool fin_new = false;  /* observables from (xn, vn) instead of (x, v) */
            double t_fin = 0.0;
            if (mode == MODE_RUN) {
                if (accept) {
                    ++steps_acc;
                    /* events (R6): sign changes of s = d.w at accepted-step ends */
                    const bool neg_old = s_old < 0.0, neg_new = s_new < 0.0;
                    if (neg_old != neg_new) {
                        ++n_tp;
                        if (neg_old && r2n < P.rcsq) {
                            const double tc = now + h * s_old / (s_old - s_new);
                            if (n_coll == 0) t_first = tc;
                            t_last = tc;
                            ++n_coll;
                        }
                    }
                    if (r2n > P.r0sq && s_new > 0.0) {
                        /* exit (R7): first upward crossing of |d| = r0; localise it by Newton on
                         * g(hk) = |d(t_n + hk)|^2 - r0^2 over uncontrolled steps from (t_n, y_n) */
                        const double g = r2n - P.r0sq;
                        if (fabs(g) <= P.loc_tol) {
                            fin = 0; fin_new = true; t_fin = now + h;
                        } else {
                            mode = MODE_LOC;
                            n_loc = 0;
                            h = h - g / (2.0 * s_new);
                        }
                    } else {
                        /* commit */
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
                        s_old = s_new;
                        if (last) {
                            fin = 1; t_fin = P.t_max;
                        } else {
                            if (!failed) h = h * fmin(5.0, 0.8 * yq);
                            if (h > P.h_max) h = P.h_max;
                            failed = false;
                        }
                    }
                } else {
                    ++steps_rej;
                    if (h <= P.h_min) {
                        fin = 2; t_fin = now;
                    } else if (!failed) {
                        failed = true;
                        h = fmax(P.h_min, h * fmax(0.1, 0.8 * yq));
                    } else {
                        h = fmax(P.h_min, 0.5 * h);
                    }
                }
                if (fin < 0 && mode == MODE_RUN &&
                    (unsigned long long)steps_acc + (unsigned long long)steps_rej >= P.max_steps) {
                    fin = 4;
                    t_fin = (double)n_per * P.T_rf + tf;
                }
            } else { /* MODE_LOC */
                ++n_loc;
                const double g = r2n - P.r0sq;
                if (fabs(g) <= P.loc_tol || n_loc >= 8) {
                    fin = 0; fin_new = true; t_fin = now + h;
                } else {
                    h = h - g / (2.0 * s_new);
                }
            }

            if (fin >= 0) {
                /* observables (R10) + record (a10) + ensemble reduction (a11) */
                const double w0 = fin_new ? vn[0] : v[0], w1 = fin_new ? vn[1] : v[1], w2 = fin_new ? vn[2] : v[2];
                const double ke = 0.5 * P.m_i * (w0 * w0 + w1 * w1 + w2 * w2);
                if (O.records != nullptr) {
                    ia_record r;
                    r.ke_ion = ke;
                    r.t_dwell = t_fin;
                    r.t_life = (n_coll >= 2) ? (t_last - t_first) : 0.0;
                    r.va_f[0] = fin_new ? vn[3] : v[3];
                    r.va_f[1] = fin_new ? vn[4] : v[4];
                    r.va_f[2] = fin_new ? vn[5] : v[5];
                    r.n_coll = n_coll;
                    r.n_tp = n_tp;
                    r.steps_acc = steps_acc;
                    r.steps_rej = (uint16_t)min(steps_rej, 65535u);
                    r.status = (uint8_t)fin;
                    r.n_loc = (uint8_t)n_loc;
                    O.records[slot] = r;
                }
                if (O.summary != nullptr) {
                    ia_summary *S = O.summary;
                    atomicAdd((unsigned long long *)&S->n_done, 1ull);
                    atomicAdd((unsigned long long *)&S->n_status[fin], 1ull);
                    if (n_coll >= 2) atomicAdd((unsigned long long *)&S->n_complex, 1ull);
                    atomicAdd((unsigned long long *)&S->steps_acc, (unsigned long long)steps_acc);
                    atomicAdd((unsigned long long *)&S->steps_rej, (unsigned long long)steps_rej);
                    atomicAdd((unsigned long long *)&S->steps_loc, (unsigned long long)n_loc);
                    if (fin == 0) {
                        atomicAdd(&S->sum_ke, ke);
                        atomicAdd(&S->sum_ke2, ke * ke);
                    }
                    const int bin = (n_coll == 0) ? 0 : min(32 - __clz(n_coll), IA_HIST_BINS - 1);
                    atomicAdd((unsigned long long *)&S->hist_ncoll[bin], 1ull);
                }
                mode = MODE_IDLE;
            }
        }
    }
    if (O.summary != nullptr && lane == 0) atomicMax((unsigned long long *)&O.summary->t_end_ns, ia_globaltimer());
}

/* ---- host launchers ------------------------------------------------------------------------ */

cudaError_t ia_launch_persistent(const IaParams &P, const IaGen &G, const IaOut &O, unsigned long long *counter,
                                 unsigned long long warn, int grid_blocks, cudaStream_t st) {
    ia_persistent_kernel<<<grid_blocks, IA_THREADS, 0, st>>>(P, G, O, counter, warn);
    return cudaGetLastError();
}

cudaError_t ia_persistent_info(int device, int *blocks_per_sm, int *threads_per_block, int *regs, int *local_bytes) {
    (void)device;
    cudaFuncAttributes fa;
    cudaError_t e = cudaFuncGetAttributes(&fa, ia_persistent_kernel);
    if (e != cudaSuccess) return e;
    int nb = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, ia_persistent_kernel, IA_THREADS, 0);
    if (e != cudaSuccess) return e;
    *blocks_per_sm = nb;
    *threads_per_block = IA_THREADS;
    *regs = fa.numRegs;
    *local_bytes = (int)fa.localSizeBytes;
    return cudaSuccess;
}

cudaError_t ia_launch_generate(const IaParams &P, const IaGen &G, double *ic_dump, cudaStream_t st) {
    const unsigned threads = 128;
    const unsigned long long blocks = (G.n + threads - 1) / threads;
    ia_generate_kernel<<<(unsigned)blocks, threads, 0, st>>>(P, G, ic_dump);
    return cudaGetLastError();
}

#define IA_VARIANT fma
#include "ia_verify.cuh"
