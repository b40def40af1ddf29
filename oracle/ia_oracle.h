/*
 * ia_oracle.h -- C interface of the CPU ORACLE for the ion+atom trajectory path of arXiv 2509.15117.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * `--impl reference` legs may load this library.  It shares no code with the CUDA path under
 * paper_2509_15117_b200/ and neither imports the other.
 *
 * Plain, slow, single-thread, first-order-form Dormand-Prince 5(4) (refs [22,23])
 * on the 12-variable system of PAPER.md:13-20 (Eq. 1-2).  See ia_oracle.cpp for the per-function
 * citations and DESIGN.md section "Readings" (R1..R18) for every point the paper leaves open.
 */
#ifndef IA_ORACLE_H
#define IA_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    double m_ion_u, m_atom_u, alpha_au; /* masses in u, polarisability in a.u.       */
    double a[3], q[3], omega_rf_au;     /* Mathieu a_k, q_k, rf angular frequency */
    double De_K, r0_a0;                 /* well depth in K (C8 = C4^2/(4 De)), start/exit sphere   */
    double rtol, atol;                  /* ode45-style tolerances (reading R5)                     */
    double t_max_rf;                    /* time limit in rf periods (reading R8)                   */
    double h_max_rf;                    /* step-size cap in rf periods                             */
    double r_coll_a0;                   /* bounce threshold (reading R6)                           */
    uint64_t max_steps;                 /* cap on attempted steps                                  */
} oracle_params;

/* quantities derived from the parameters, all in atomic units */
typedef struct {
    double m_i, m_a, C4, C8, De, r_e, Omega, T_rf, thr, h_max, h_min, t_max, r0, r_coll;
} oracle_derived;

typedef struct {
    double ke_ion, t_dwell, t_life, va_f[3];  /* same meaning as the GPU record                      */
    uint32_t n_coll, n_tp, steps_acc, steps_rej, n_loc;
    int32_t status;                           /* 0 escaped, 1 t_max, 2 h<h_min, 3 non-finite, 4 max_steps */
    double y_final[12];                       /* r_i, r_a, v_i, v_a at termination                   */
    double t_first, t_last;                   /* first / last short-range collision times            */
    double h_first, h_last;                   /* initial step size, last attempted step size         */
} oracle_outcome;

/* initial-condition generator description (mirrors the launch descriptor of the boundary) */
typedef struct {
    int32_t mode;                 /* 1 = GRID, 2 = PHILOX, 3 = THERMAL (0 = explicit is not generated) */
    int32_t domain;               /* 0 octant, 1 full sphere                              */
    int32_t phase_mode;           /* 0 fixed phase0, 1 uniform in [0,2pi) from Philox      */
    uint32_t n_theta, n_phi;      /* GRID                                                  */
    double phase0;
    double E_min_uK, E_max_uK;    /* equal: fixed energy; else log-uniform from Philox     */
    uint64_t seed; uint32_t cell; uint64_t first_index;
    double T_atom_uK, T_ion_uK;   /* THERMAL (reading R18): bath and ion temperatures */
} oracle_gen;

int  oracle_derive(const oracle_params *p, oracle_derived *d);
/* V(r) = C8/r^8 - C4/r^4 */
double oracle_potential(const oracle_params *p, double r);
/* f(t,y): t_frac is the time folded into one rf period, phase the rf phase at t = 0 */
void oracle_rhs(const oracle_params *p, double t_frac, double phase, const double y[12], double f[12]);
/* one uncontrolled DP5(4) step of size h; e = error estimate vector (may be NULL) */
void oracle_step(const oracle_params *p, double t_frac, double phase, const double y[12], double h,
                 double ynew[12], double e[12]);
/* ode45 error norm of a step, max_i |e_i| / max(|y_i|,|ynew_i|,atol/rtol) */
double oracle_err_norm(const oracle_params *p, const double y[12], const double ynew[12], const double e[12]);
/* nsteps uncontrolled steps of size h; states is [nsteps+1][13] = (t, y) rows */
void oracle_trace(const oracle_params *p, const double y0[12], double phase, double h, uint32_t nsteps,
                  double *states);
/* adaptive run to termination. path (may be NULL) receives (t, y[12]) rows of accepted steps,
 * at most path_cap rows; *path_len receives how many were written. */
int  oracle_run(const oracle_params *p, const double y0[12], double phase, oracle_outcome *out,
                double *path, uint64_t path_cap, uint64_t *path_len);
/* Philox4x32-10 */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* reading R2: the uniform deviate in (0,1] made of two Philox words */
double oracle_u53(uint32_t w_even, uint32_t w_odd);
/* generate trajectory `index` (local index; global = first_index + index): y0[12], phase, E (E_h) */
int  oracle_generate(const oracle_params *p, const oracle_gen *g, uint64_t index, double y0[12],
                     double *phase, double *E_au);
/* run `count` generated trajectories, local indices indices[i] (or first + i when indices is NULL),
 * farmed over nthreads std::threads (one trajectory per task; the integrator stays single-threaded). */
int  oracle_run_generated(const oracle_params *p, const oracle_gen *g, const uint64_t *indices, uint64_t first,
                          uint64_t count, oracle_outcome *outs, int nthreads);
/* same for explicit initial conditions y0[count][12], phase[count] */
int  oracle_run_explicit(const oracle_params *p, const double *y0, const double *phase, uint64_t count,
                         oracle_outcome *outs, int nthreads);
/* the tableau as the oracle holds it: c[7], a[7][7] (row-major, lower triangle), b[7], bhat[7] */
void oracle_tableau(double c[7], double a[49], double b[7], double bhat[7]);

#ifdef __cplusplus
}
#endif
#endif
