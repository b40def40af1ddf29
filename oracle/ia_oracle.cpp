/*
 * ia_oracle.cpp -- CPU ORACLE for the ion+atom trajectory path of arXiv 2509.15117.
 *
 * TEST INFRASTRUCTURE ONLY (see ia_oracle.h).  Plain C++17, single thread per trajectory, FP64,
 * built with -O2 -ffp-contract=off so every operation is an individually rounded IEEE operation.
 * It follows the method step by step, in first-order form on the 12-vector
 *     y = (r_i[3], r_a[3], v_i[3], v_a[3])
 * with no blocking, fusion or reordering:
 *   - right-hand side: Newton's equations of H, Eq. 1-2 with
 *     V(r) = C8/r^8 - C4/r^4, C4 = alpha/2, C8 = C4^2/(4 De) (BASELINE.json north_star);
 *   - pair: Dormand-Prince 5(4), 7 stages, FSAL, local extrapolation (ref [22]);
 *   - controller: the ode45 scheme of ref [23], reading R5;
 *   - events, termination, exit localisation, observables: DESIGN.md readings R6-R10
 *     (the paper names the observables at PAPER.md:24,30 but not how they are detected);
 *   - initial conditions: head-on runs, grid / Philox sampling (readings R1-R3).
 *
 * Parity pins (tests/test_oracle_*.py): tableau order conditions, potential minimum and depth,
 * force = -grad V, Newton's third law, z-axis harmonic period, Mathieu characteristic exponent,
 * classical deflection integral, energy / angular momentum / linear momentum conservation,
 * mirror symmetry, convergence order, Philox known-answer vectors, the word -> uniform map and the GRID / PHILOX
 * direction, phase and energy maps, the error norm and every branch of the step-size law on a linear problem with
 * a closed-form step, the collision times against the turning-point quadrature (tests/test_oracle_pins2.py).
 * Unpinned: none of the paper's figure values are recoverable (images absent), so the ensemble
 * statistics (P(complex), histograms) are "parity unpinned" against the paper -- only trend checks.
 */
#include "ia_oracle.h"

#include <atomic>
#include <cmath>
#include <cstring>
#include <limits>
#include <thread>
#include <vector>

namespace {

/* CODATA 2022 conversion factors (values; the CUDA path carries its own copy) */
const double ME_PER_U = 1822.888486283;      /* electron masses per atomic mass unit */
const double KB_EH_PER_K = 3.1668115634564e-6; /* Boltzmann constant in Hartree per kelvin */
const double PI = 3.14159265358979323846;

struct Derived {
    double m_i, m_a, C4, C8, De, r_e, Omega, T_rf, thr, h_max, h_min, t_max, r0, r_coll;
    double a[3], q[3];
    double rtol, atol, t_max_rf;
    uint64_t max_steps;
};

Derived derive(const oracle_params &p) {
    Derived D;
    D.m_i = p.m_ion_u * ME_PER_U;
    D.m_a = p.m_atom_u * ME_PER_U;
    D.C4 = p.alpha_au / 2.0;
    D.De = p.De_K * KB_EH_PER_K;
    D.C8 = D.C4 * D.C4 / (4.0 * D.De);             /* north_star: C8 = C4^2/(4 De) */
    D.r_e = std::pow(2.0 * D.C8 / D.C4, 0.25);     /* V'(r_e) = 0 */
    D.Omega = p.omega_rf_au;
    D.T_rf = 2.0 * PI / D.Omega;
    D.rtol = p.rtol;
    D.atol = p.atol;
    D.thr = p.atol / p.rtol;                       /* ode45 threshold, reading R5 */
    D.h_max = p.h_max_rf * D.T_rf;
    D.h_min = std::ldexp(D.T_rf, -40);             /* reading R5: h_min = 2^-40 T_rf */
    D.t_max_rf = p.t_max_rf;
    D.t_max = p.t_max_rf * D.T_rf;
    D.r0 = p.r0_a0;
    D.r_coll = p.r_coll_a0;
    for (int k = 0; k < 3; ++k) { D.a[k] = p.a[k]; D.q[k] = p.q[k]; }
    D.max_steps = p.max_steps;
    return D;
}

/* Dormand-Prince 5(4) tableau, ref [22]; SURVEY.md section 8(c)-O3 lists it. */
const double C[7] = {0.0, 1.0 / 5.0, 3.0 / 10.0, 4.0 / 5.0, 8.0 / 9.0, 1.0, 1.0};
const double A[7][7] = {
    {0, 0, 0, 0, 0, 0, 0},
    {1.0 / 5.0, 0, 0, 0, 0, 0, 0},
    {3.0 / 40.0, 9.0 / 40.0, 0, 0, 0, 0, 0},
    {44.0 / 45.0, -56.0 / 15.0, 32.0 / 9.0, 0, 0, 0, 0},
    {19372.0 / 6561.0, -25360.0 / 2187.0, 64448.0 / 6561.0, -212.0 / 729.0, 0, 0, 0},
    {9017.0 / 3168.0, -355.0 / 33.0, 46732.0 / 5247.0, 49.0 / 176.0, -5103.0 / 18656.0, 0, 0},
    {35.0 / 384.0, 0.0, 500.0 / 1113.0, 125.0 / 192.0, -2187.0 / 6784.0, 11.0 / 84.0, 0}};
const double B[7] = {35.0 / 384.0, 0.0, 500.0 / 1113.0, 125.0 / 192.0, -2187.0 / 6784.0, 11.0 / 84.0, 0.0};
const double BHAT[7] = {5179.0 / 57600.0, 0.0, 7571.0 / 16695.0, 393.0 / 640.0,
                        -92097.0 / 339200.0, 187.0 / 2100.0, 1.0 / 40.0};

/* O1: f(t,y).  t_frac is time folded into [0,T_rf) (reading R9); the trap term
 * uses cos(Omega t + phase) with t counted from the start of the run (reading R3). */
void rhs(const Derived &D, double t_frac, double phase, const double y[12], double f[12]) {
    const double *ri = y, *ra = y + 3, *vi = y + 6, *va = y + 9;
    double d[3];
    double r2 = 0.0;
    for (int k = 0; k < 3; ++k) {
        d[k] = ra[k] - ri[k];
        r2 += d[k] * d[k];
    }
    const double u = 1.0 / r2;
    /* force on the atom = -dV/dr * d/r = (8 C8 r^-10 - 4 C4 r^-6) d */
    const double s = u * u * u * (8.0 * D.C8 * u * u - 4.0 * D.C4);
    const double c = std::cos(D.Omega * t_frac + phase);
    for (int k = 0; k < 3; ++k) {
        f[k] = vi[k];
        f[3 + k] = va[k];
        /* ion: reaction of the pair force + Paul-trap force -(a_k + 2 q_k cos) m_i Omega^2/4 r_k */
        f[6 + k] = -(s / D.m_i) * d[k] - (D.a[k] + 2.0 * D.q[k] * c) * (D.Omega * D.Omega / 4.0) * ri[k];
        f[9 + k] = (s / D.m_a) * d[k];
    }
}

/* One DP5(4) step from (t_frac, y) with k1 = f(t,y) given.  Writes the 5th-order solution ynew,
 * k7 = f(t+h, ynew) (FSAL) and the error estimate e = h * sum_l (b_l - bhat_l) k_l. */
void dp5_step(const Derived &D, double t_frac, double phase, const double y[12], const double k1[12],
              double h, double ynew[12], double k7[12], double e[12]) {
    double k[7][12];
    std::memcpy(k[0], k1, sizeof(double) * 12);
    double ys[12];
    for (int s = 1; s < 7; ++s) {
        for (int i = 0; i < 12; ++i) {
            double acc = 0.0;
            for (int l = 0; l < s; ++l) acc += A[s][l] * k[l][i];
            ys[i] = y[i] + h * acc;
        }
        rhs(D, t_frac + C[s] * h, phase, ys, k[s]);
        if (s == 6) std::memcpy(ynew, ys, sizeof(double) * 12); /* row 7 of A is b: ys is y_{n+1} */
    }
    std::memcpy(k7, k[6], sizeof(double) * 12);
    for (int i = 0; i < 12; ++i) {
        double acc = 0.0;
        for (int l = 0; l < 7; ++l) acc += (B[l] - BHAT[l]) * k[l][i];
        e[i] = h * acc;
    }
}

/* reading R5: err = max_i |e_i| / max(|y_i|, |ynew_i|, atol/rtol) */
double err_norm(const Derived &D, const double y[12], const double ynew[12], const double e[12]) {
    double err = 0.0;
    bool bad = false;
    for (int i = 0; i < 12; ++i) {
        double sc = std::fmax(std::fmax(std::fabs(y[i]), std::fabs(ynew[i])), D.thr);
        double r = std::fabs(e[i]) / sc;
        if (std::isnan(r)) bad = true;
        else if (r > err) err = r;
    }
    return bad ? std::numeric_limits<double>::quiet_NaN() : err;
}

inline void sep(const double y[12], double *r2, double *s) {
    double rr = 0.0, ss = 0.0;
    for (int k = 0; k < 3; ++k) {
        const double d = y[3 + k] - y[k];
        const double w = y[9 + k] - y[6 + k];
        rr += d * d;
        ss += d * w;
    }
    *r2 = rr;
    *s = ss;
}

bool all_finite(const double y[12]) {
    for (int i = 0; i < 12; ++i)
        if (!std::isfinite(y[i])) return false;
    return true;
}

void finish(const Derived &D, oracle_outcome *out, int status, const double y[12], double t,
            double t_first, double t_last) {
    out->status = status;
    const double *vi = y + 6, *va = y + 9;
    out->ke_ion = 0.5 * D.m_i * (vi[0] * vi[0] + vi[1] * vi[1] + vi[2] * vi[2]); /* R10 */
    out->t_dwell = t;
    out->t_first = t_first;
    out->t_last = t_last;
    out->t_life = (out->n_coll >= 2) ? (t_last - t_first) : 0.0;                    /* R6 */
    for (int k = 0; k < 3; ++k) out->va_f[k] = va[k];
    std::memcpy(out->y_final, y, sizeof(double) * 12);
}

/* O4: one trajectory, adaptive, to termination. */
int run_one(const Derived &D, const double y0[12], double phase, oracle_outcome *out, double *path,
            uint64_t path_cap, uint64_t *path_len) {
    std::memset(out, 0, sizeof(*out));
    uint64_t np = 0;
    double y[12];
    std::memcpy(y, y0, sizeof(y));
    uint64_t n_per = 0; /* completed rf periods (reading R9) */
    double tf = 0.0;    /* time folded into [0, T_rf) */
    double t_first = 0.0, t_last = 0.0;
    auto now = [&]() { return (double)n_per * D.T_rf + tf; };
    auto record = [&](double t, const double *yy) {
        if (path && np < path_cap) {
            path[np * 13] = t;
            std::memcpy(path + np * 13 + 1, yy, sizeof(double) * 12);
            ++np;
        }
        if (path_len) *path_len = np;
    };
    record(0.0, y);
    if (!all_finite(y) || !std::isfinite(phase)) {
        finish(D, out, 3, y, 0.0, 0.0, 0.0);
        return 0;
    }
    double k1[12];
    rhs(D, tf, phase, y, k1);
    /* initial step, reading R5 (ode45): h = min(h_max, t_max); rho = ||f0/max(|y0|,thr)||_inf /
     * (0.8 rtol^(1/5)); if h rho > 1, h = 1/rho */
    double h = std::fmin(D.h_max, D.t_max);
    {
        double rho = 0.0;
        for (int i = 0; i < 12; ++i) {
            double r = std::fabs(k1[i]) / std::fmax(std::fabs(y[i]), D.thr);
            if (r > rho) rho = r;
        }
        rho = rho / (0.8 * std::pow(D.rtol, 0.2));
        if (h * rho > 1.0) h = 1.0 / rho;
        if (h < D.h_min) h = D.h_min;
    }
    out->h_first = h;
    double r2_old, s_old;
    sep(y, &r2_old, &s_old);
    bool failed = false; /* a rejection has happened since the last accepted step */
    uint64_t attempts = 0;
    const double r0sq = D.r0 * D.r0;
    const double rcsq = D.r_coll * D.r_coll;
    for (;;) {
        /* clip the last step to land on t_max (reading R5/R8) */
        bool last = false;
        {
            const double rem = (D.t_max_rf - (double)n_per) * D.T_rf - tf;
            if (h >= rem) {
                h = rem;
                last = true;
            }
        }
        double ynew[12], k7[12], e[12];
        dp5_step(D, tf, phase, y, k1, h, ynew, k7, e);
        const double err = err_norm(D, y, ynew, e);
        ++attempts;
        out->h_last = h;
        if (err <= D.rtol) {
            /* ---- accepted ---- */
            out->steps_acc++;
            double r2_new, s_new;
            sep(ynew, &r2_new, &s_new);
            /* events, reading R6: sign changes of s = d.w sampled at accepted-step ends */
            const bool neg_old = (s_old < 0.0), neg_new = (s_new < 0.0);
            if (neg_old != neg_new) {
                out->n_tp++;
                if (neg_old && r2_new < rcsq) { /* minimum of r(t) at short range: a bounce */
                    const double tc = now() + h * s_old / (s_old - s_new);
                    if (out->n_coll == 0) t_first = tc;
                    t_last = tc;
                    out->n_coll++;
                }
            }
            /* exit, reading R7: first upward crossing of |d| = r0 */
            if (r2_new > r0sq && s_new > 0.0) {
                /* localise: Newton on g(hk) = |d(t_n + hk)|^2 - r0^2 over uncontrolled steps from
                 * (t_n, y_n), until |g| <= 1e-13 r0^2.  Reading R7 as amended: the iterate is kept inside the
                 * bracket [lo, hi] (g(hi) > 0 known, lo = 0 where the trajectory was still inside): a Newton
                 * proposal that leaves it -- a near-tangential exit, d.w ~ 0 -- is replaced by the midpoint;
                 * otherwise one uncontrolled step of many rf periods can blow the ion's state up.  At most
                 * 60 iterations (a bracket of 2^-60 h). */
                double hk = h, g = r2_new - r0sq;
                double lo = 0.0, hi = h;
                uint32_t nloc = 0;
                /* a trajectory that was already outside at t_n (a thermal start beyond r0 that never came in)
                 * has no crossing to localise: it ends with the detecting step */
                while (r2_old < r0sq && std::fabs(g) > 1e-13 * r0sq && nloc < 60) {
                    if (nloc > 0) {
                        if (g > 0.0) hi = hk; else lo = hk;
                    }
                    double hn = hk - g / (2.0 * s_new);
                    if (!(s_new > 0.0 && hn > lo && hn < hi)) hn = 0.5 * (lo + hi);
                    hk = hn;
                    dp5_step(D, tf, phase, y, k1, hk, ynew, k7, e);
                    sep(ynew, &r2_new, &s_new);
                    g = r2_new - r0sq;
                    ++nloc;
                }
                out->n_loc = nloc;
                out->steps_rej = (uint32_t)(attempts - out->steps_acc);
                if (!all_finite(ynew)) {
                    /* R7: a localisation step that is not finite (it only shortens a finite accepted step, so this is
                     * not reachable from finite states) is not an escape: status 3 at the last state inside */
                    finish(D, out, 3, y, now(), t_first, t_last);
                    return 0;
                }
                const double t_exit = now() + hk;
                record(t_exit, ynew);
                finish(D, out, 0, ynew, t_exit, t_first, t_last);
                return 0;
            }
            /* commit */
            tf += h;
            if (tf >= D.T_rf) {
                tf -= D.T_rf;
                ++n_per;
            }
            std::memcpy(y, ynew, sizeof(y));
            std::memcpy(k1, k7, sizeof(k1));
            s_old = s_new;
            r2_old = r2_new;
            record(now(), y);
            if (last) {
                out->steps_rej = (uint32_t)(attempts - out->steps_acc);
                finish(D, out, 1, y, D.t_max, t_first, t_last);
                return 0;
            }
            if (!failed) {
                const double f = 1.25 * std::pow(err / D.rtol, 0.2);
                h = (f > 0.2) ? h / f : 5.0 * h;
            }
            if (h > D.h_max) h = D.h_max;
            failed = false;
        } else {
            /* ---- rejected ---- */
            if (h <= D.h_min) {
                out->steps_rej = (uint32_t)(attempts - out->steps_acc);
                finish(D, out, 2, y, now(), t_first, t_last);
                return 0;
            }
            if (!failed) {
                failed = true;
                double fac = 0.1;
                if (std::isfinite(err)) fac = std::fmax(0.1, 0.8 * std::pow(D.rtol / err, 0.2));
                h = std::fmax(D.h_min, h * fac);
            } else {
                h = std::fmax(D.h_min, 0.5 * h);
            }
        }
        if (attempts >= D.max_steps) {
            out->steps_rej = (uint32_t)(attempts - out->steps_acc);
            finish(D, out, 4, y, now(), t_first, t_last);
            return 0;
        }
    }
}

/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), written from the published round function:
 * multipliers 0xD2511F53, 0xCD9E8D57; Weyl key increments 0x9E3779B9, 0xBB67AE85. */
void philox(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n1 = (uint32_t)p1;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        const uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* reading R2: uniform in (0,1] from two words: (k + 1/2) 2^-53 with the 53-bit integer k = (we >> 5) 2^26 + (wo >> 6),
 * the sum k + 1/2 rounded to double (exact below k = 2^52, ties-to-even from there on, so the largest k gives 1.0) */
double u53(uint32_t we, uint32_t wo) {
    return ((double)(we >> 5) * 67108864.0 + (double)(wo >> 6) + 0.5) * (1.0 / 9007199254740992.0);
}

int generate(const Derived &D, const oracle_gen &g, uint64_t index, double y0[12], double *phase,
             double *E_au) {
    const uint64_t gi = g.first_index + index;
    uint32_t key[2] = {(uint32_t)g.seed, (uint32_t)(g.seed >> 32)};
    uint32_t ctr[4] = {(uint32_t)gi, (uint32_t)(gi >> 32), g.cell, 0u};
    uint32_t w0[4], w1[4];
    philox(ctr, key, w0);
    ctr[3] = 1u;
    philox(ctr, key, w1);
    const double u1 = u53(w0[0], w0[1]), u2 = u53(w0[2], w0[3]);
    const double u3 = u53(w1[0], w1[1]), u4 = u53(w1[2], w1[3]);
    double ct, st, phi;
    if (g.mode == 1) { /* GRID, reading R1: cell-centred, uniform in theta and phi */
        if (g.n_theta == 0 || g.n_phi == 0) return -1;
        const uint64_t i = index / g.n_phi, j = index % g.n_phi;
        const double th_span = (g.domain == 0) ? PI / 2.0 : PI;
        const double ph_span = (g.domain == 0) ? PI / 2.0 : 2.0 * PI;
        const double theta = ((double)i + 0.5) * th_span / (double)g.n_theta;
        phi = ((double)j + 0.5) * ph_span / (double)g.n_phi;
        ct = std::cos(theta);
        st = std::sin(theta);
    } else if (g.mode == 2) { /* PHILOX, reading R2 */
        if (g.domain == 0) {
            ct = u1;
            phi = (PI / 2.0) * u2;
        } else {
            ct = 2.0 * u1 - 1.0;
            phi = 2.0 * PI * u2;
        }
        st = std::sqrt(1.0 - ct * ct);
    } else if (g.mode == 3) {
        /* THERMAL (reading R18).  Atom: uniform on the sphere of radius r0 about the trap
         * centre, Cartesian velocity components Gaussian with variance k_B T/m_a, "negated if needed to enforce
         * v_r < 0".  Ion: position and momentum Gaussian "corresponding to a fixed temperature ... for a spherical
         * harmonic trap with frequency omega = q_x Omega_rf / 2^(3/2)".  Normal deviates by Box-Muller on the
         * Philox blocks 2..6: (z_2k, z_2k+1) = sqrt(-2 ln u_a) (cos 2 pi u_b, sin 2 pi u_b). */
        if (!(g.T_atom_uK > 0.0) || !(g.T_ion_uK > 0.0) || D.q[0] == 0.0) return -1;
        ct = 2.0 * u1 - 1.0;
        phi = 2.0 * PI * u2;
        st = std::sqrt(1.0 - ct * ct);
        double z[10];
        for (uint32_t b = 2; b <= 6; ++b) {
            uint32_t w[4];
            ctr[3] = b;
            philox(ctr, key, w);
            const double ua = u53(w[0], w[1]), ub = u53(w[2], w[3]);
            const double R = std::sqrt(-2.0 * std::log(ua));
            z[2 * (b - 2)] = R * std::cos(2.0 * PI * ub);
            z[2 * (b - 2) + 1] = R * std::sin(2.0 * PI * ub);
        }
        const double kT_i = g.T_ion_uK * 1e-6 * KB_EH_PER_K, kT_a = g.T_atom_uK * 1e-6 * KB_EH_PER_K;
        const double w_h = std::fabs(D.q[0]) * D.Omega / std::pow(2.0, 1.5);
        const double s_v = std::sqrt(kT_i / D.m_i), s_r = s_v / w_h, s_a = std::sqrt(kT_a / D.m_a);
        const double n[3] = {st * std::cos(phi), st * std::sin(phi), ct};
        double va[3], vr = 0.0;
        for (int k = 0; k < 3; ++k) {
            va[k] = s_a * z[6 + k];
            vr += va[k] * n[k];
        }
        const double sign = (vr > 0.0) ? -1.0 : 1.0;
        double v2 = 0.0;
        for (int k = 0; k < 3; ++k) {
            y0[k] = s_r * z[k];
            y0[3 + k] = D.r0 * n[k];
            y0[6 + k] = s_v * z[3 + k];
            y0[9 + k] = sign * va[k];
            v2 += va[k] * va[k];
        }
        *phase = (g.phase_mode == 1) ? 2.0 * PI * u3 : g.phase0;
        *E_au = 0.5 * D.m_a * v2;
        return 0;
    } else {
        return -1;
    }
    *phase = (g.phase_mode == 1) ? 2.0 * PI * u3 : g.phase0;
    double E_uK = g.E_min_uK;
    if (g.E_max_uK != g.E_min_uK) E_uK = g.E_min_uK * std::pow(g.E_max_uK / g.E_min_uK, u4);
    const double E = E_uK * 1e-6 * KB_EH_PER_K;
    *E_au = E;
    const double v0 = std::sqrt(2.0 * E / D.m_a); /* E = m_a v0^2 / 2 */
    const double n[3] = {st * std::cos(phi), st * std::sin(phi), ct};
    for (int k = 0; k < 3; ++k) {
        y0[k] = 0.0;            /* ion at the trap centre */
        y0[3 + k] = D.r0 * n[k]; /* atom on the sphere of radius r0 */
        y0[6 + k] = 0.0;        /* ion at rest */
        y0[9 + k] = -v0 * n[k]; /* atom aimed at the ion */
    }
    return 0;
}

template <class F>
void farm(uint64_t count, int nthreads, F f) {
    if (nthreads < 1) nthreads = 1;
    if ((uint64_t)nthreads > count) nthreads = (int)(count ? count : 1);
    std::atomic<uint64_t> next(0);
    auto worker = [&]() {
        for (;;) {
            const uint64_t i = next.fetch_add(1);
            if (i >= count) break;
            f(i);
        }
    };
    if (nthreads == 1) {
        worker();
        return;
    }
    std::vector<std::thread> th;
    for (int t = 0; t < nthreads; ++t) th.emplace_back(worker);
    for (auto &t : th) t.join();
}

} // namespace

extern "C" {

int oracle_derive(const oracle_params *p, oracle_derived *d) {
    if (!p || !d) return -1;
    const Derived D = derive(*p);
    d->m_i = D.m_i; d->m_a = D.m_a; d->C4 = D.C4; d->C8 = D.C8; d->De = D.De; d->r_e = D.r_e;
    d->Omega = D.Omega; d->T_rf = D.T_rf; d->thr = D.thr; d->h_max = D.h_max; d->h_min = D.h_min;
    d->t_max = D.t_max; d->r0 = D.r0; d->r_coll = D.r_coll;
    return 0;
}

double oracle_potential(const oracle_params *p, double r) {
    const Derived D = derive(*p);
    return D.C8 / std::pow(r, 8) - D.C4 / std::pow(r, 4);
}

void oracle_rhs(const oracle_params *p, double t_frac, double phase, const double y[12], double f[12]) {
    rhs(derive(*p), t_frac, phase, y, f);
}

void oracle_step(const oracle_params *p, double t_frac, double phase, const double y[12], double h,
                 double ynew[12], double e[12]) {
    const Derived D = derive(*p);
    double k1[12], k7[12], ee[12];
    rhs(D, t_frac, phase, y, k1);
    dp5_step(D, t_frac, phase, y, k1, h, ynew, k7, ee);
    if (e) std::memcpy(e, ee, sizeof(ee));
}

double oracle_err_norm(const oracle_params *p, const double y[12], const double ynew[12], const double e[12]) {
    return err_norm(derive(*p), y, ynew, e);
}

void oracle_trace(const oracle_params *p, const double y0[12], double phase, double h, uint32_t nsteps,
                  double *states) {
    const Derived D = derive(*p);
    double y[12], k1[12], ynew[12], k7[12], e[12];
    std::memcpy(y, y0, sizeof(y));
    uint64_t n_per = 0;
    double tf = 0.0;
    states[0] = 0.0;
    std::memcpy(states + 1, y, sizeof(y));
    rhs(D, tf, phase, y, k1);
    for (uint32_t n = 0; n < nsteps; ++n) {
        dp5_step(D, tf, phase, y, k1, h, ynew, k7, e);
        tf += h;
        if (tf >= D.T_rf) {
            tf -= D.T_rf;
            ++n_per;
        }
        std::memcpy(y, ynew, sizeof(y));
        std::memcpy(k1, k7, sizeof(k1));
        states[(uint64_t)(n + 1) * 13] = (double)n_per * D.T_rf + tf;
        std::memcpy(states + (uint64_t)(n + 1) * 13 + 1, y, sizeof(y));
    }
}

int oracle_run(const oracle_params *p, const double y0[12], double phase, oracle_outcome *out,
               double *path, uint64_t path_cap, uint64_t *path_len) {
    if (!p || !y0 || !out) return -1;
    return run_one(derive(*p), y0, phase, out, path, path_cap, path_len);
}

void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    philox(ctr, key, out);
}

double oracle_u53(uint32_t w_even, uint32_t w_odd) { return u53(w_even, w_odd); }

int oracle_generate(const oracle_params *p, const oracle_gen *g, uint64_t index, double y0[12],
                    double *phase, double *E_au) {
    if (!p || !g || !y0 || !phase || !E_au) return -1;
    return generate(derive(*p), *g, index, y0, phase, E_au);
}

int oracle_run_generated(const oracle_params *p, const oracle_gen *g, const uint64_t *indices, uint64_t first,
                         uint64_t count, oracle_outcome *outs, int nthreads) {
    if (!p || !g || !outs) return -1;
    const Derived D = derive(*p);
    std::atomic<int> bad(0);
    farm(count, nthreads, [&](uint64_t i) {
        double y0[12], phase, E;
        if (generate(D, *g, indices ? indices[i] : first + i, y0, &phase, &E) != 0) {
            bad = 1;
            return;
        }
        run_one(D, y0, phase, &outs[i], nullptr, 0, nullptr);
    });
    return bad ? -1 : 0;
}

int oracle_run_explicit(const oracle_params *p, const double *y0, const double *phase, uint64_t count,
                        oracle_outcome *outs, int nthreads) {
    if (!p || !y0 || !phase || !outs) return -1;
    const Derived D = derive(*p);
    farm(count, nthreads, [&](uint64_t i) { run_one(D, y0 + 12 * i, phase[i], &outs[i], nullptr, 0, nullptr); });
    return 0;
}

void oracle_tableau(double c[7], double a[49], double b[7], double bhat[7]) {
    for (int i = 0; i < 7; ++i) {
        c[i] = C[i];
        b[i] = B[i];
        bhat[i] = BHAT[i];
        for (int j = 0; j < 7; ++j) a[i * 7 + j] = A[i][j];
    }
}

} // extern "C"
