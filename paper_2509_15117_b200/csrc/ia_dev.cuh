/*
 * ia_dev.cuh -- device arithmetic of the ion+atom propagator: right-hand side, one Dormand-Prince
 * 5(4) attempt in second-order (Nystrom-collapsed) form, error norm, fifth root, cosine.
 *
 * Included by ia_kernels.cu (production arithmetic, FMA contraction on) and by ia_nofma.cu
 * (compiled with -fmad=false: every a*b+c below is two rounded operations there; only the explicit
 * fma() calls in the reciprocal / range reduction stay fused).  Shares nothing with oracle/.
 *
 * Method (Eq. 1-2, PAPER.md:20,26 refs [22,23]):
 *   y = (x, v) with x = (r_i, r_a), v = (v_i, v_a); dx/dt = v, dv/dt = A(t, x) -- the force does not
 *   depend on velocity, so the 7-stage DP5(4) step collapses exactly to
 *       X_s   = x + (h c_s) v + h^2 sum_l abar_sl A_l,      abar = a.a
 *       v_new = v + h sum_l b_l A_l,        x_new = X_7
 *       e_x   = h^2 sum_l ebar_l A_l,       e_v = h sum_l E_l A_l,   ebar = E.a,  E = b - bhat
 *   (sum_l E_l = 0 removes the v term of e_x).  The stage velocities V_2..V_6 are never formed.
 */
#pragma once
#include <stdint.h>

struct IaParams {
    /* pair potential and masses */
    double inv_m_a;     /*  1/m_a                       */
    double neg_inv_m_i; /* -1/m_i                       */
    double m_i, m_a;
    double c8x8, c4x4;  /* 8 C8, 4 C4                   */
    /* trap: A_i,k += (ka_k + kq_k cos(Omega t + phase)) r_i,k */
    double ka[3];       /* -a_k Omega^2/4               */
    double kq[3];       /* -q_k Omega^2/2               */
    double omega, T_rf;
    /* controller (reading R5) */
    double rtol, thr, inv_rtol;
    double h_max, h_min, t_max_rf, t_max;
    double h0_scale;    /* 0.8 rtol^(1/5) (divides rho) */
    /* events / termination (R6, R7) */
    double r0, r0sq, rcsq, loc_tol; /* loc_tol = 1e-13 r0^2 */
    double C4, C8, De, r_e, r_coll, atol;
    unsigned long long max_steps;
};

#define IA_DEV __device__ __forceinline__

/* ---- small FP64 helpers ------------------------------------------------------------------- */

/* 1/x for normal, finite, non-zero x: MUFU.RCP64H seed (rel. err <= 2^-23) and one third-order
 * correction y <- y + y(e + e^2), e = 1 - x y  (error e^3 ~ 2^-69, result within ~1 ulp).
 * x = 0, inf or NaN gives NaN -- the callers rely on that to flag non-finite states. */
IA_DEV double ia_rcp(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    const double e2 = fma(e, e, e);
    return fma(y, e2, y);
}

/* x^(-1/5) for x in [1e-30, 1e30]: FP32 MUFU seed (lg2/ex2, rel. err ~1e-6) and two Newton steps
 * y <- y (6 - x y^5)/5 (rel. err -> 3e-12 -> ~3e-23). */
IA_DEV double ia_inv_fifth_root(double x) {
    const float xf = (float)x;
    float lf;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(lf) : "f"(xf));
    float sf;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(sf) : "f"(-0.2f * lf));
    double y = (double)sf;
#pragma unroll
    for (int it = 0; it < 2; ++it) {
        const double y2 = y * y;
        const double y4 = y2 * y2;
        const double y5 = y4 * y;
        const double t = fma(-x, y5, 6.0);
        y = (0.2 * y) * t;
    }
    return y;
}

/* cos(arg) for arg in about [-4 pi, 8 pi] (the callers keep time folded, reading R9):
 * n = rint(arg/pi), r = arg - n pi (two-constant Cody-Waite with exact fma products),
 * cos(arg) = (-1)^n cos(r), |r| <= pi/2, Taylor polynomial in r^2 through r^22
 * (truncation (pi/2)^24/24! = 8e-20; absolute error ~1e-16). */
IA_DEV double ia_cos_folded(double arg) {
    const double MAGIC = 6755399441055744.0; /* 1.5 * 2^52: adding it rounds to nearest integer */
    const double nf = fma(arg, 0.31830988618379067154, MAGIC);
    const double n = nf - MAGIC;
    double r = fma(-n, 3.14159265358979311600e+00, arg);
    r = fma(-n, 1.22464679914735317723e-16, r);
    const double z = r * r;
    double p = -1.0 / 1124000727777607680000.0;          /* -1/22! */
    p = p * z + 1.0 / 2432902008176640000.0;             /*  1/20! */
    p = p * z - 1.0 / 6402373705728000.0;                /* -1/18! */
    p = p * z + 1.0 / 20922789888000.0;                  /*  1/16! */
    p = p * z - 1.0 / 87178291200.0;                     /* -1/14! */
    p = p * z + 1.0 / 479001600.0;                       /*  1/12! */
    p = p * z - 1.0 / 3628800.0;                         /* -1/10! */
    p = p * z + 1.0 / 40320.0;                           /*  1/8!  */
    p = p * z - 1.0 / 720.0;                             /* -1/6!  */
    p = p * z + 1.0 / 24.0;                              /*  1/4!  */
    p = p * z - 0.5;                                     /* -1/2!  */
    p = p * z + 1.0;
    /* flip the sign when n is odd: the integer n sits in the low word of nf */
    const int lo = __double2loint(nf);
    const int hi = __double2hiint(p) ^ (lo << 31);
    return __hiloint2double(hi, __double2loint(p));
}

/* ---- right-hand side (reading O1) ------------------------------------------ */

/* Accelerations A[0..2] (ion) and A[3..5] (atom) at positions X = (r_i, r_a), with c = cos(Omega t
 * + phase).  Also returns r^2 = |r_a - r_i|^2 and the scalar s = u^3 (8 C8 u^2 - 4 C4), u = 1/r^2:
 * force on the atom = -dV/dr d/r = s d. */
IA_DEV void ia_accel(const IaParams &P, const double (&X)[6], double c, double (&A)[6], double &r2, double &s) {
    const double d0 = X[3] - X[0], d1 = X[4] - X[1], d2 = X[5] - X[2];
    r2 = d0 * d0 + d1 * d1 + d2 * d2;
    const double u = ia_rcp(r2);
    const double u2 = u * u;
    const double t = P.c8x8 * u2 - P.c4x4;
    s = (u2 * u) * t;
    const double sa = s * P.inv_m_a;
    const double si = s * P.neg_inv_m_i;
    A[3] = sa * d0;
    A[4] = sa * d1;
    A[5] = sa * d2;
    A[0] = si * d0 + (P.ka[0] + P.kq[0] * c) * X[0];
    A[1] = si * d1 + (P.ka[1] + P.kq[1] * c) * X[1];
    A[2] = si * d2 + (P.ka[2] + P.kq[2] * c) * X[2];
}

/* ---- Dormand-Prince 5(4), ref [22] ------------------------------------------- */
/* nodes */
#define IA_C2 (1.0 / 5.0)
#define IA_C3 (3.0 / 10.0)
#define IA_C4 (4.0 / 5.0)
#define IA_C5 (8.0 / 9.0)
/* abar = a.a (exact rationals; tests/test_host_logic.py re-derives them from the tableau) */
#define IA_AB31 (9.0 / 200.0)
#define IA_AB41 (-12.0 / 25.0)
#define IA_AB42 (4.0 / 5.0)
#define IA_AB51 (-12248.0 / 6561.0)
#define IA_AB52 (7208.0 / 2187.0)
#define IA_AB53 (-6784.0 / 6561.0)
#define IA_AB61 (-533.0 / 264.0)
#define IA_AB62 (91.0 / 22.0)
#define IA_AB63 (-56.0 / 33.0)
#define IA_AB64 (7.0 / 88.0)
#define IA_AB71 (35.0 / 384.0)
#define IA_AB73 (50.0 / 159.0)
#define IA_AB74 (25.0 / 192.0)
#define IA_AB75 (-243.0 / 6784.0)
/* b (5th-order weights; b2 = b7 = 0) */
#define IA_B1 (35.0 / 384.0)
#define IA_B3 (500.0 / 1113.0)
#define IA_B4 (125.0 / 192.0)
#define IA_B5 (-2187.0 / 6784.0)
#define IA_B6 (11.0 / 84.0)
/* E = b - bhat (E2 = 0) */
#define IA_E1 (71.0 / 57600.0)
#define IA_E3 (-71.0 / 16695.0)
#define IA_E4 (71.0 / 1920.0)
#define IA_E5 (-17253.0 / 339200.0)
#define IA_E6 (22.0 / 525.0)
#define IA_E7 (-1.0 / 40.0)
/* ebar = E.a (ebar2 = ebar7 = 0) */
#define IA_EB1 (611.0 / 230400.0)
#define IA_EB3 (-514.0 / 83475.0)
#define IA_EB4 (391.0 / 38400.0)
#define IA_EB5 (-4617.0 / 1356800.0)
#define IA_EB6 (-11.0 / 3360.0)

struct IaErr {
    double num, den; /* err = num/den = max_i |e_i| / max(|y_i|, |ynew_i|, thr)   (reading R5) */
};

/* keeps the larger of two ratios na/da, nb/db (all >= 0, denominators > 0) by cross-multiplication */
IA_DEV void ia_ratio_max(double &na, double &da, double nb, double db) {
    const bool gt = nb * da > na * db;
    na = gt ? nb : na;
    da = gt ? db : da;
}

/* One uncontrolled DP5(4) step of size h from (tf, x, v) with A1 = A(tf, x) given.
 * Out: xn, vn (5th-order solution), A7 = A(tf + h, xn) (FSAL), r2n = |d(xn)|^2, the error-norm
 * argmax pair, and finite = false when the step produced a non-finite separation. */
IA_DEV void ia_dp5_attempt(const IaParams &P, const double (&x)[6], const double (&v)[6], const double (&A1)[6],
                           double tf, double phase, double h, double (&xn)[6], double (&vn)[6],
                           double (&A7)[6], double &r2n, IaErr &err, bool &finite) {
    const double hh = h * h;
    double X[6], A2[6], A3[6], A4[6], A5[6], A6[6];
    double r2, s;
    /* stage 2 */
    {
        const double hc = h * IA_C2;
#pragma unroll
        for (int i = 0; i < 6; ++i) X[i] = x[i] + hc * v[i];
        const double c = ia_cos_folded(P.omega * (tf + hc) + phase);
        ia_accel(P, X, c, A2, r2, s);
    }
    /* stage 3 */
    {
        const double hc = h * IA_C3, g1 = hh * IA_AB31;
#pragma unroll
        for (int i = 0; i < 6; ++i) X[i] = x[i] + hc * v[i] + g1 * A1[i];
        const double c = ia_cos_folded(P.omega * (tf + hc) + phase);
        ia_accel(P, X, c, A3, r2, s);
    }
    /* stage 4 */
    {
        const double hc = h * IA_C4, g1 = hh * IA_AB41, g2 = hh * IA_AB42;
#pragma unroll
        for (int i = 0; i < 6; ++i) X[i] = x[i] + hc * v[i] + g1 * A1[i] + g2 * A2[i];
        const double c = ia_cos_folded(P.omega * (tf + hc) + phase);
        ia_accel(P, X, c, A4, r2, s);
    }
    /* stage 5 */
    {
        const double hc = h * IA_C5, g1 = hh * IA_AB51, g2 = hh * IA_AB52, g3 = hh * IA_AB53;
#pragma unroll
        for (int i = 0; i < 6; ++i) X[i] = x[i] + hc * v[i] + g1 * A1[i] + g2 * A2[i] + g3 * A3[i];
        const double c = ia_cos_folded(P.omega * (tf + hc) + phase);
        ia_accel(P, X, c, A5, r2, s);
    }
    /* stages 6 and 7 share the time t + h, hence the cosine */
    const double c1 = ia_cos_folded(P.omega * (tf + h) + phase);
    {
        const double g1 = hh * IA_AB61, g2 = hh * IA_AB62, g3 = hh * IA_AB63, g4 = hh * IA_AB64;
#pragma unroll
        for (int i = 0; i < 6; ++i) X[i] = x[i] + h * v[i] + g1 * A1[i] + g2 * A2[i] + g3 * A3[i] + g4 * A4[i];
        ia_accel(P, X, c1, A6, r2, s);
    }
    /* 5th-order solution: x_new = X_7, v_new = v + h sum b_l A_l */
    {
        const double g1 = hh * IA_AB71, g3 = hh * IA_AB73, g4 = hh * IA_AB74, g5 = hh * IA_AB75;
        const double w1 = h * IA_B1, w3 = h * IA_B3, w4 = h * IA_B4, w5 = h * IA_B5, w6 = h * IA_B6;
#pragma unroll
        for (int i = 0; i < 6; ++i) {
            xn[i] = x[i] + h * v[i] + g1 * A1[i] + g3 * A3[i] + g4 * A4[i] + g5 * A5[i];
            vn[i] = v[i] + w1 * A1[i] + w3 * A3[i] + w4 * A4[i] + w5 * A5[i] + w6 * A6[i];
        }
        ia_accel(P, xn, c1, A7, r2n, s);
    }
    finite = (s == s); /* s is NaN whenever r2 of stage 7 is 0, inf or NaN (see ia_rcp) */
    /* error estimate and ode45 norm (R5) */
    {
        const double q1 = hh * IA_EB1, q3 = hh * IA_EB3, q4 = hh * IA_EB4, q5 = hh * IA_EB5, q6 = hh * IA_EB6;
        const double p1 = h * IA_E1, p3 = h * IA_E3, p4 = h * IA_E4, p5 = h * IA_E5, p6 = h * IA_E6, p7 = h * IA_E7;
        double en[12], sc[12];
#pragma unroll
        for (int i = 0; i < 6; ++i) {
            const double ex = q1 * A1[i] + q3 * A3[i] + q4 * A4[i] + q5 * A5[i] + q6 * A6[i];
            const double ev = p1 * A1[i] + p3 * A3[i] + p4 * A4[i] + p5 * A5[i] + p6 * A6[i] + p7 * A7[i];
            en[i] = fabs(ex);
            en[6 + i] = fabs(ev);
            sc[i] = fmax(fmax(fabs(x[i]), fabs(xn[i])), P.thr);
            sc[6 + i] = fmax(fmax(fabs(v[i]), fabs(vn[i])), P.thr);
        }
        /* tree of cross-multiplied comparisons */
#pragma unroll
        for (int i = 0; i < 6; ++i) ia_ratio_max(en[i], sc[i], en[6 + i], sc[6 + i]);
#pragma unroll
        for (int i = 0; i < 3; ++i) ia_ratio_max(en[i], sc[i], en[3 + i], sc[3 + i]);
        ia_ratio_max(en[0], sc[0], en[1], sc[1]);
        ia_ratio_max(en[0], sc[0], en[2], sc[2]);
        err.num = en[0];
        err.den = sc[0];
    }
}

/* d.w with d = r_a - r_i, w = v_a - v_i: sign of dr/dt (reading R6) */
IA_DEV double ia_sdot(const double (&x)[6], const double (&v)[6]) {
    return (x[3] - x[0]) * (v[3] - v[0]) + (x[4] - x[1]) * (v[4] - v[1]) + (x[5] - x[2]) * (v[5] - v[2]);
}
