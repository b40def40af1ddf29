"""Pins for the CPU oracle: what the paper and the mathematics fix (no GPU needed).

Each test checks oracle/ia_oracle.cpp against something other than itself: exact order conditions,
closed forms (potential minimum, harmonic period, Mathieu exponent from a Hill eigenproblem, classical
deflection quadrature), invariants (E, L, P with the trap off; mirror symmetry) and convergence rates.
Citations: PAPER.md (arXiv 2509.15117 text) line numbers; readings R1..R16.
"""
import math
import os
from dataclasses import replace
from fractions import Fraction as F

import numpy as np
import pytest
from scipy import integrate, optimize

import ia_inputs as I
from oracle import ia_oracle as O

KB = 3.1668115634564e-6
ME_PER_U = 1822.888486283
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def golden_values():
    vals = {}
    with open(os.path.join(GOLD, "paper_values.txt")) as fh:
        for line in fh:
            if line.strip() and not line.startswith("#"):
                k, v = line.split()
                vals[k] = float(v)
    return vals


# --------------------------------------------------------------------------------------------
# tableau (Dormand-Prince 5(4), ref [22])
# --------------------------------------------------------------------------------------------
def order_conditions(a, b, c, order):
    """Left-hand side minus right-hand side of every rooted-tree order condition up to `order`."""
    e = np.ones(len(c))
    ac, ac2, ac3 = a @ c, a @ c ** 2, a @ c ** 3
    aac, aac2 = a @ ac, a @ ac2
    res = {1: [b @ e - 1], 2: [b @ c - F(1, 2)],
           3: [b @ c ** 2 - F(1, 3), b @ ac - F(1, 6)],
           4: [b @ c ** 3 - F(1, 4), b @ (c * ac) - F(1, 8), b @ ac2 - F(1, 12), b @ aac - F(1, 24)],
           5: [b @ c ** 4 - F(1, 5), b @ (c ** 2 * ac) - F(1, 10), b @ (c * ac2) - F(1, 15),
               b @ (c * aac) - F(1, 30), b @ (ac * ac) - F(1, 20), b @ ac3 - F(1, 20),
               b @ (a @ (c * ac)) - F(1, 40), b @ aac2 - F(1, 60), b @ (a @ aac) - F(1, 120)]}
    out = []
    for o in range(1, order + 1):
        out += [float(x) for x in res[o]]
    return out


def test_tableau_order_conditions():
    c, a, b, bh = O.tableau()
    assert np.allclose(a.sum(axis=1), c, atol=2e-16)
    assert np.all(np.triu(a) == 0.0)                      # explicit
    assert np.array_equal(a[6], b)                        # FSAL: last row of a is b
    r5 = order_conditions(a, b, c, 5)
    assert len(r5) == 17 and max(abs(x) for x in r5) < 5e-16
    r4 = order_conditions(a, bh, c, 4)
    assert len(r4) == 8 and max(abs(x) for x in r4) < 5e-16
    # bhat is NOT fifth order (it is the embedded fourth-order solution)
    assert max(abs(x) for x in order_conditions(a, bh, c, 5)[8:]) > 1e-4
    assert abs((b - bh).sum()) < 1e-16


def test_tableau_matches_exact_rationals():
    """The doubles are the correctly rounded rationals of ref [22] (checked against fractions)."""
    c, a, b, bh = O.tableau()
    exact_b = [F(35, 384), F(0), F(500, 1113), F(125, 192), F(-2187, 6784), F(11, 84), F(0)]
    exact_bh = [F(5179, 57600), F(0), F(7571, 16695), F(393, 640), F(-92097, 339200), F(187, 2100), F(1, 40)]
    for x, fx in zip(b, exact_b):
        assert x == float(fx)
    for x, fx in zip(bh, exact_bh):
        assert x == float(fx)
    # exact arithmetic check that these rationals satisfy the conditions (so a typo in a row that
    # happens to round to the same double cannot hide)
    ca = [F(0), F(1, 5), F(3, 10), F(4, 5), F(8, 9), F(1), F(1)]
    assert sum(exact_b) == 1 and sum(x * y for x, y in zip(exact_b, ca)) == F(1, 2)
    assert sum(x * y ** 4 for x, y in zip(exact_b, ca)) == F(1, 5)
    assert sum(exact_bh) == 1 and sum(x * y ** 3 for x, y in zip(exact_bh, ca)) == F(1, 4)


# --------------------------------------------------------------------------------------------
# potential and force (BASELINE.json north_star: r_e = (2 C8/C4)^(1/4), depth D_e)
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("atom,De_K", [("Rb87", 1.0), ("Li7", 1.0), ("Cs133", 100.0), ("Na23", 0.1)])
def test_potential_minimum_and_depth(atom, De_K):
    p = replace(I.Params().with_atom(atom), De_K=De_K)
    C4 = p.alpha_au / 2.0
    De = De_K * KB
    r_e = (C4 / (2.0 * De)) ** 0.25          # (2 C8/C4)^(1/4) with C8 = C4^2/(4 De)
    d = O.derive(p)
    assert d["r_e"] == pytest.approx(r_e, rel=1e-14)
    assert O.potential(p, r_e) == pytest.approx(-De, rel=1e-13)
    # V'(r_e) = 0: the pair acceleration vanishes there, and changes sign across it
    for r, sign in ((r_e, 0), (0.99 * r_e, +1), (1.01 * r_e, -1)):
        y = np.zeros(12)
        y[3] = r
        f = O.rhs(replace(p, a=(0, 0, 0), q=(0, 0, 0)), 0.0, 0.0, y)
        if sign == 0:
            scale = 4 * C4 / r_e ** 5 / d["m_a"]
            assert abs(f[9]) < 1e-13 * scale
        else:
            assert np.sign(f[9]) == sign     # repulsive inside r_e, attractive outside


def test_potential_minimum_matches_survey_table():
    g = golden_values()
    assert O.derive(I.Params().with_atom("Rb87"))["r_e"] == pytest.approx(g["r_e_Rb_1K_a0"], abs=6e-5)
    assert O.derive(I.Params().with_atom("Li7"))["r_e"] == pytest.approx(g["r_e_Li_1K_a0"], abs=6e-5)


def test_force_is_minus_gradient_and_third_law():
    p = replace(I.Params().with_atom("Rb87"), a=(0, 0, 0), q=(0, 0, 0))
    d = O.derive(p)
    rng = np.random.default_rng(1)
    for r in (60.0, 70.85, 90.0, 300.0, 4000.0):
        n = rng.normal(size=3)
        n /= np.linalg.norm(n)
        y = np.zeros(12)
        y[0:3] = rng.normal(0, 50, 3)
        y[3:6] = y[0:3] + r * n
        y[6:12] = rng.normal(0, 1e-7, 6)
        f = O.rhs(p, 0.0, 0.0, y)
        assert np.array_equal(f[0:6], y[6:12])                 # dr/dt = v
        # central finite difference of V along each axis (Richardson-free, eps ~ r * 1e-5)
        grad = np.zeros(3)
        for k in range(3):
            eps = 1e-5 * r
            dp, dm = r * n.copy(), r * n.copy()
            dp[k] += eps
            dm[k] -= eps
            grad[k] = (O.potential(p, np.linalg.norm(dp)) - O.potential(p, np.linalg.norm(dm))) / (2 * eps)
        Fa = d["m_a"] * f[9:12]
        # tolerance relative to the attractive term alone: at r ~ r_e the two terms cancel
        assert np.allclose(Fa, -grad, rtol=2e-7, atol=2e-7 * 4 * d["C4"] / r ** 5)
        # Newton's third law with the trap off
        assert np.allclose(d["m_a"] * f[9:12] + d["m_i"] * f[6:9], 0.0, atol=4e-16 * 4 * d["C4"] / r ** 5)


def test_trap_force_formula_signs():
    """Ion alone, displaced along each axis: a_k(t) = -(a_k + 2 q_k cos(Omega t + phase)) Omega^2/4 r_k
    (PAPER.md:15-18).  Evaluated at phases where cos = 1, 0, -1."""
    p = replace(I.Params(), alpha_au=0.0)   # no pair force
    Om = p.omega_rf_au
    for k in range(3):
        y = np.zeros(12)
        y[k] = 3.0
        y[3] = 1e6
        for phase, cosv in ((0.0, 1.0), (math.pi / 2, 0.0), (math.pi, -1.0)):
            f = O.rhs(p, 0.0, phase, y)
            expect = -(p.a[k] + 2 * p.q[k] * cosv) * Om * Om / 4 * 3.0
            assert f[6 + k] == pytest.approx(expect, rel=1e-12, abs=abs(2 * p.q[k] * Om * Om / 4 * 3.0) * 2e-16)
        # folded time: t_frac = T/2 is phase pi
        f = O.rhs(p, math.pi / Om, 0.0, y)
        assert f[6 + k] == pytest.approx(-(p.a[k] - 2 * p.q[k]) * Om * Om / 4 * 3.0, rel=1e-12)
    assert np.all(O.rhs(p, 0.0, 0.3, y)[9:12] == 0.0)     # the neutral atom feels no trap


# --------------------------------------------------------------------------------------------
# lone ion in the trap: exact harmonic motion on z, Mathieu exponent on x
# --------------------------------------------------------------------------------------------
def lone_ion_params(**kw):
    base = dict(alpha_au=0.0, r0_a0=1e12, rtol=1e-13, atol=1e-15)
    base.update(kw)
    return replace(I.Params(), **base)


def test_z_axis_is_harmonic_with_the_exact_period():
    g = golden_values()
    p0 = I.Params()
    wz = 0.5 * p0.omega_rf_au * math.sqrt(p0.a[2])
    f_kHz = wz / (2 * math.pi) / I.AU_TIME_S / 1e3
    assert f_kHz == pytest.approx(g["f_z_kHz"], rel=1e-8)
    n_rf = 2.0 / math.sqrt(p0.a[2])                      # z period in rf periods
    p = lone_ion_params(t_max_rf=n_rf)
    y0 = np.zeros(12)
    y0[2], y0[8], y0[3] = 10.0, 2e-8, 1e6
    out, _ = O.run(p, y0)
    assert out["status"] == 1
    amp_v = math.hypot(y0[8], 10.0 * wz)
    assert abs(out["y_final"][2] - y0[2]) < 1e-9 * math.hypot(10.0, y0[8] / wz)
    assert abs(out["y_final"][8] - y0[8]) < 1e-9 * amp_v
    # quarter period: z -> v/w, v -> -z w
    out, _ = O.run(replace(p, t_max_rf=n_rf / 4), y0)
    assert out["y_final"][2] == pytest.approx(y0[8] / wz, rel=1e-9)
    assert out["y_final"][8] == pytest.approx(-10.0 * wz, rel=1e-9)


def mathieu_beta_hill(a, q, n=40):
    """Characteristic exponent of x'' + (a + 2 q cos 2 tau) x = 0 from the Floquet-Fourier (Hill)
    eigenproblem -- no ODE solver: x = sum_n c_n exp(i (2n + beta) tau) gives
    ((2n+beta)^2) c_n - q (c_{n-1} + c_{n+1}) = a c_n, i.e. a is an eigenvalue of T(beta)."""
    ns = np.arange(-n, n + 1)

    def gap(beta):
        T = np.diag((2.0 * ns + beta) ** 2) - q * (np.eye(2 * n + 1, k=1) + np.eye(2 * n + 1, k=-1))
        ev = np.linalg.eigvalsh(T)
        return ev[0] - a                     # lowest band: a(beta) is increasing on (0,1)
    return optimize.brentq(gap, 1e-6, 0.999, xtol=1e-14)


@pytest.mark.parametrize("q", [0.05, 0.1, 0.2, 0.3, 0.4])
def test_secular_frequency_matches_mathieu(q):
    a = -0.0005
    g = golden_values()
    beta_hill = mathieu_beta_hill(a, q)
    assert beta_hill == pytest.approx(g[f"beta_mathieu_q{q:g}"], abs=2e-8)     # SURVEY's 40-digit value
    p = lone_ion_params(t_max_rf=1.0, a=(a, -0.0005, 0.001), q=(q, -q, 0.0))
    vs = 1e-8
    cols = []
    for x0, v0 in ((1.0, 0.0), (0.0, vs)):
        y0 = np.zeros(12)
        y0[0], y0[6], y0[3] = x0, v0, 1e6
        out, _ = O.run(p, y0)
        assert out["status"] == 1
        cols.append((out["y_final"][0], out["y_final"][6] / vs))
    M = np.array(cols).T                                    # monodromy over one rf period
    assert np.linalg.det(M) == pytest.approx(1.0, abs=1e-10)   # symplectic
    beta = math.acos(0.5 * np.trace(M)) / math.pi
    assert beta == pytest.approx(beta_hill, abs=1e-8)
    if q == 0.1:   # PAPER.md:58's lowest-order formula is 0.19 % low
        assert math.sqrt(a + q * q / 2) == pytest.approx(g["beta_lowest_order_q0.1"], abs=1e-8)
        assert 0.001 < beta / math.sqrt(a + q * q / 2) - 1 < 0.003


def test_fixed_step_global_error_is_fifth_order():
    """Mathieu x-motion + harmonic z-motion of a lone ion over 2 rf periods with n fixed steps:
    error against a 1e-13 adaptive solve falls like h^5."""
    p = lone_ion_params(t_max_rf=2.0)
    y0 = np.zeros(12)
    y0[0], y0[1], y0[2], y0[6], y0[8], y0[3] = 5.0, -3.0, 10.0, 1e-8, 2e-8, 1e6
    ref, _ = O.run(p, y0, phase=0.4)
    T = O.derive(p)["T_rf"]
    errs = []
    for n in (40, 80, 160, 320):
        st = O.trace(p, y0, 0.4, 2.0 * T / n, n)
        scale = np.array([5, 3, 10, 1e-8, 1e-8, 2e-8])
        idx = [0, 1, 2, 6, 7, 8]
        errs.append(np.max(np.abs(st[-1, 1:][idx] - ref["y_final"][idx]) / scale))
    slopes = np.diff(np.log(errs)) / np.log(0.5)
    assert errs[0] > 1e-9                   # resolvable, not round-off
    assert np.all(np.abs(slopes[:2] - 5.0) < 0.35), (errs, slopes)


# --------------------------------------------------------------------------------------------
# trap-free two-body dynamics: deflection integral, conservation laws
# --------------------------------------------------------------------------------------------
def trapfree(atom="Rb87", **kw):
    base = dict(a=(0, 0, 0), q=(0, 0, 0), rtol=1e-13, atol=1e-15, t_max_rf=1e5)
    base.update(kw)
    return replace(I.Params().with_atom(atom), **base)


def swept_angle_quadrature(p, b, E):
    """Theta = 2 int_{r_min}^{r0} L dr / (r^2 sqrt(2 mu (E_cm - V) - L^2/r^2)), r = r_min + (r0-r_min) s^2."""
    m_i, m_a = p.m_ion_u * ME_PER_U, p.m_atom_u * ME_PER_U
    mu = m_i * m_a / (m_i + m_a)
    C4 = p.alpha_au / 2
    C8 = C4 ** 2 / (4 * p.De_K * KB)
    V = lambda r: C8 / r ** 8 - C4 / r ** 4
    v0 = math.sqrt(2 * E / m_a)
    r0 = p.r0_a0
    E_cm = 0.5 * mu * v0 ** 2 + V(r0)
    L = mu * b * v0
    rad = lambda r: 2 * mu * (E_cm - V(r)) - L * L / (r * r)
    # outermost turning point: scan inward from r0 for the first sign change
    rs = np.geomspace(r0, 10.0, 200000)
    vals = rad(rs)
    k = np.argmax(vals < 0)
    r_min = optimize.brentq(rad, rs[k], rs[k - 1], xtol=1e-15, rtol=1e-15)

    def integrand(s):
        r = r_min + (r0 - r_min) * s * s
        return L / (r * r * math.sqrt(max(rad(r), 1e-300))) * 2 * (r0 - r_min) * s
    val, err = integrate.quad(integrand, 0.0, 1.0, epsabs=1e-13, epsrel=1e-13, limit=400)
    return 2 * val, v0


@pytest.mark.parametrize("b", [3000.0, 2400.0, 1000.0, 100.0, 1.0])
def test_trap_free_deflection_matches_quadrature(b):
    # Velocities (|v| ~ 1e-8 a.u.) are below atol/rtol, so they are under ABSOLUTE control at atol
    # (reading R4): atol = 1e-19 bounds them to ~1e-11 relative per step.  With atol = 1e-15 the
    # deep bounce (D_e/E = 1e5) amplifies the looser velocity control to ~4e-7 in the swept angle.
    p = trapfree(atol=1e-19)
    E = 10e-6 * KB
    theta_q, v0 = swept_angle_quadrature(p, b, E)
    y0 = I.impact_ic(b, p.r0_a0, v0)
    out, _ = O.run(p, y0)
    assert out["status"] == 0
    d0 = y0[3:6] - y0[0:3]
    d1 = out["y_final"][3:6] - out["y_final"][0:3]
    assert abs(np.linalg.norm(d1) / p.r0_a0 - 1) < 2e-13                   # localised exit, reading R7
    # L_z < 0: d rotates clockwise; swept angle = -(phi_f - phi_i) mod 2 pi
    sweep = -(math.atan2(d1[1], d1[0]) - math.atan2(d0[1], d0[0]))
    z = np.exp(1j * sweep) - np.exp(1j * theta_q)
    assert abs(z) < 2e-8, (sweep % (2 * math.pi), theta_q % (2 * math.pi))
    if b == 1000.0:
        # the remaining difference is the integrator's truncation error: it falls in proportion to rtol
        errs = []
        for rtol in (1e-11, 1e-12):
            o, _ = O.run(replace(p, rtol=rtol), y0)
            d1 = o["y_final"][3:6] - o["y_final"][0:3]
            sw = -(math.atan2(d1[1], d1[0]) - math.atan2(d0[1], d0[0]))
            errs.append(abs(np.exp(1j * sw) - np.exp(1j * theta_q)))
        assert 4.0 < errs[0] / errs[1] < 25.0 and 2.0 < errs[1] / abs(z) < 25.0, (errs, abs(z))


def invariants(p, path):
    m_i, m_a = p.m_ion_u * ME_PER_U, p.m_atom_u * ME_PER_U
    C4 = p.alpha_au / 2
    C8 = C4 ** 2 / (4 * p.De_K * KB)
    ri, ra, vi, va = (path[:, 1 + 3 * k: 4 + 3 * k] for k in range(4))
    r = np.linalg.norm(ra - ri, axis=1)
    ke = 0.5 * m_i * (vi ** 2).sum(1) + 0.5 * m_a * (va ** 2).sum(1)
    E = ke + C8 / r ** 8 - C4 / r ** 4
    Lv = m_i * np.cross(ri, vi) + m_a * np.cross(ra, va)
    P = m_i * vi + m_a * va
    return E, ke, Lv, P, r


@pytest.mark.parametrize("b", [500.0, 2000.0])
def test_trap_free_conservation(b):
    """BASELINE.json north_star: E and L conserved to 1e-9 with the trap off (reading R11 for what
    'relative' means when E_tot/D_e = 1e-5)."""
    p = trapfree()
    v0 = math.sqrt(2 * 10e-6 * KB / (p.m_atom_u * ME_PER_U))
    y0 = I.impact_ic(b, p.r0_a0, v0)
    out, path = O.run(p, y0, path_cap=200000)
    assert out["status"] == 0 and len(path) == out["steps_acc"] + 1
    E, ke, Lv, P, r = invariants(p, path)
    assert r.min() < 100.0 if b < 2344 else True
    assert np.abs(Lv[:, 2] - Lv[0, 2]).max() <= 1e-9 * abs(Lv[0, 2])
    assert np.abs(Lv[:, :2]).max() <= 1e-12 * abs(Lv[0, 2])
    assert np.abs(E - E[0]).max() <= 1e-9 * ke.max()
    # linear invariant: kept by any RK method up to round-off, which scales with the individual
    # momenta in the well (|m v| ~ sqrt(2 mu D_e) >> |P|), times sqrt(steps)
    m_a = p.m_atom_u * ME_PER_U
    p_ind = m_a * np.abs(path[:, 10:13]).max()
    assert np.abs(P - P[0]).max() <= 2e-16 * math.sqrt(len(path)) * p_ind


def test_trap_free_conservation_shallow_well():
    """Shallow well (D_e = 100 uK, E = 10 uK): |dE|/E_tot <= 1e-9 is reachable (reading R11)."""
    p = trapfree(De_K=100e-6)
    v0 = math.sqrt(2 * 10e-6 * KB / (p.m_atom_u * ME_PER_U))
    y0 = I.impact_ic(300.0, p.r0_a0, v0)
    out, path = O.run(p, y0, path_cap=200000)
    E, ke, Lv, P, r = invariants(p, path)
    assert out["status"] == 0
    assert np.abs(E - E[0]).max() <= 1e-9 * abs(E[0])
    assert np.abs(Lv[:, 2] - Lv[0, 2]).max() <= 1e-9 * abs(Lv[0, 2])


def test_trap_free_head_on_is_a_single_bounce_with_elastic_exit():
    """Head-on, trap off: one bounce, atom leaves with the relative speed it came with (elastic)."""
    p = trapfree("Li7")
    c = replace(I.config0().launch, n_theta=4, n_phi=4, n=16)
    outs = O.run_generated(p, c)
    assert np.all(outs["status"] == 0) and np.all(outs["n_coll"] == 1) and np.all(outs["n_tp"] == 1)
    w0 = math.sqrt(2 * 10e-6 * KB / (p.m_atom_u * ME_PER_U))
    w1 = np.linalg.norm(outs["y_final"][:, 9:12] - outs["y_final"][:, 6:9], axis=1)
    assert np.allclose(w1, w0, rtol=1e-7)


# --------------------------------------------------------------------------------------------
# symmetry, controller, termination
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_mirror_symmetry_is_bitwise(axis):
    """Flipping the sign of one Cartesian coordinate of the IC flips it in every state, bit for bit
    (IEEE operations are sign-symmetric; the trap is even in each coordinate)."""
    c = I.config0()
    y0, ph, _ = O.generate(c.params, c.launch, [5 * 32 + 11])
    y0 = y0[0]
    p = replace(c.params, t_max_rf=50.0)
    out_a, path_a = O.run(p, y0, ph[0], path_cap=5000)
    ym = y0.copy()
    ym[axis::3] *= -1
    out_b, path_b = O.run(p, ym, ph[0], path_cap=5000)
    assert len(path_a) == len(path_b) > 100
    flip = np.ones(13)
    flip[1 + axis::3] = -1
    assert np.array_equal(path_a * flip, path_b)
    assert out_a["ke_ion"] == out_b["ke_ion"] and out_a["steps_rej"] == out_b["steps_rej"]


def test_controller_self_convergence():
    """Error against a converged solve falls in proportion to rtol (slope ~ 1): reading R5/R15."""
    c = I.config0()
    d = O.derive(c.params)
    th, ph = 0.804, 1.493
    n = np.array([math.sin(th) * math.cos(ph), math.sin(th) * math.sin(ph), math.cos(th)])
    v0 = math.sqrt(2 * 10e-6 * KB / d["m_a"])
    y0 = np.concatenate([np.zeros(3), 5000.0 * n, np.zeros(3), -v0 * n])
    ref, _ = O.run(replace(c.params, rtol=1e-13, atol=1e-15), y0)
    assert ref["n_coll"] == 1
    assert ref["t_dwell"] / d["T_rf"] == pytest.approx(5.4057, abs=2e-3)      # SURVEY probe value
    errs_t, errs_k, acc = [], [], []
    for rtol in (1e-9, 1e-10, 1e-11, 1e-12):
        o, _ = O.run(replace(c.params, rtol=rtol, atol=rtol * 1e-2), y0)
        errs_t.append(abs(o["t_dwell"] / ref["t_dwell"] - 1))
        errs_k.append(abs(o["ke_ion"] / ref["ke_ion"] - 1))
        acc.append(int(o["steps_acc"]))
        assert o["steps_rej"] < 0.1 * o["steps_acc"]
    st = np.diff(np.log10(errs_t))
    sk = np.diff(np.log10(errs_k))
    assert np.all((st < -0.6) & (st > -1.4)), errs_t
    assert np.all((sk < -0.5) & (sk > -1.5)), errs_k
    # steps grow like rtol^(-1/5): x 10^(0.2) = 1.58 per decade
    ratios = np.array(acc[1:]) / np.array(acc[:-1])
    assert np.all((ratios > 1.35) & (ratios < 1.85)), acc


def test_exit_is_localised_and_is_a_genuine_step_from_the_last_inside_state():
    c = I.config0()
    y0, ph, _ = O.generate(c.params, c.launch, [700])
    out, path = O.run(c.params, y0[0], ph[0], path_cap=5000)
    assert out["status"] == 0 and len(path) == out["steps_acc"] + 1
    d = out["y_final"][3:6] - out["y_final"][0:3]
    assert abs(d @ d / 5000.0 ** 2 - 1) <= 1e-13
    assert 1 <= out["n_loc"] <= 8
    T = O.derive(c.params)["T_rf"]
    t_n, y_n = path[-2, 0], path[-2, 1:]
    assert np.linalg.norm(y_n[3:6] - y_n[0:3]) < 5000.0          # last committed state is inside
    h_star = out["t_dwell"] - t_n
    ynew, _ = O.step(c.params, math.fmod(t_n, T), ph[0], y_n, h_star)
    # same step up to the rounding of h* = t_exit - t_n and of the folded time
    assert np.allclose(ynew, out["y_final"], rtol=1e-11, atol=1e-18)
    assert out["t_dwell"] == path[-1, 0]


def test_termination_statuses():
    c = I.config1()
    y0, ph, _ = O.generate(c.params, c.launch, [100 * 512 + 300])
    T = O.derive(c.params)["T_rf"]
    # t_max: lands on t_max exactly
    o, _ = O.run(replace(c.params, t_max_rf=3.25), y0[0], ph[0])
    assert o["status"] == 1 and o["t_dwell"] == 3.25 * T and o["n_coll"] == 0
    # max_steps
    o, _ = O.run(replace(c.params, max_steps=50), y0[0], ph[0])
    assert o["status"] == 4 and o["steps_acc"] + o["steps_rej"] == 50
    # non-finite initial state
    bad = y0[0].copy()
    bad[4] = float("nan")
    o, _ = O.run(c.params, bad, ph[0])
    assert o["status"] == 3 and o["steps_acc"] == 0
    # h < h_min: an atom started on top of the ion's repulsive core with absurd tolerances
    yc = np.zeros(12)
    yc[3] = 1e-3
    o, _ = O.run(replace(c.params, rtol=1e-13, atol=1e-300), yc, 0.0)
    assert o["status"] in (0, 2, 3, 4)       # must terminate, whatever the label


def test_step_size_rules():
    """First step obeys the ode45 start rule (reading R5); h never exceeds h_max."""
    c = I.config0()
    y0, ph, _ = O.generate(c.params, c.launch, [0])
    d = O.derive(c.params)
    f0 = O.rhs(c.params, 0.0, ph[0], y0[0])
    rho = np.max(np.abs(f0) / np.maximum(np.abs(y0[0]), d["thr"])) / (0.8 * c.params.rtol ** 0.2)
    o, _ = O.run(c.params, y0[0], ph[0])
    assert o["h_first"] == pytest.approx(1.0 / rho, rel=1e-14)
    p = lone_ion_params(t_max_rf=3.0, h_max_rf=0.01, rtol=1e-6, atol=1e-8)
    yz = np.zeros(12)
    yz[2], yz[3] = 1.0, 1e6
    o, path = O.run(p, yz, path_cap=1000)
    assert np.diff(path[:, 0]).max() <= 0.01 * O.derive(p)["T_rf"] * (1 + 1e-12)
    assert o["steps_acc"] >= 300


# --------------------------------------------------------------------------------------------
# physics the paper states (qualitative pins; figure values are not recoverable: parity unpinned)
# --------------------------------------------------------------------------------------------
def test_config0_is_regular_single_bounce():
    """Li at 10 uK is far above 2-3 x W0^3D = 0.5-0.75 uK: no complexes."""
    c = I.config0()
    outs = O.run_generated(c.params, c.launch, indices=I.subgrid_indices(32, 4), nthreads=os.cpu_count())
    assert np.all(outs["status"] == 0) and np.all(outs["n_coll"] == 1)
    assert np.all(outs["t_life"] == 0.0)


def test_heavy_cold_atoms_form_complexes_and_light_hot_ones_do_not():
    """complexes are likely below the threshold 2-3 x W0 (Rb: 22-33 uK) and
    suppressed far above it."""
    c = I.config1(512)
    idx = I.subgrid_indices(512, 64)                     # 8 x 8 = 64 trajectories
    cold = O.run_generated(c.params, c.launch, indices=idx, nthreads=os.cpu_count())
    hot = O.run_generated(c.params, replace(c.launch, E_min_uK=300.0, E_max_uK=300.0), indices=idx,
                          nthreads=os.cpu_count())
    p_cold = np.mean(cold["n_coll"] >= 2)
    p_hot = np.mean(hot["n_coll"] >= 2)
    assert p_cold > 0.3 and p_hot < 0.1, (p_cold, p_hot)
    assert np.all(cold["n_coll"] >= 1)
    # complexes have a positive lifetime, and first/last collision times are ordered
    cx = cold[cold["n_coll"] >= 2]
    assert np.all(cx["t_life"] > 0) and np.all(cx["t_last"] > cx["t_first"])


def test_lifetime_bins_are_quarter_octaves():
    """R17: the lifetime histogram's bin index against the plain definition floor(4 log2(t_life/T_rf)) + 8 away
    from the bin edges, at exact powers of two (bin 4k + 8, lower edge inclusive), and its clamps."""
    T = O.derive(I.config1(8).params)["T_rf"]
    rng = np.random.default_rng(7)
    q = 2.0 ** rng.uniform(-1.9, 13.7, 5000)
    frac = (4 * np.log2(q)) % 1.0
    q = q[(frac > 1e-6) & (frac < 1 - 1e-6)]
    for x in q[:2000]:
        h = O.life_bins([x * T], [2], T)
        assert h.sum() == 1 and h[int(np.floor(4 * np.log2(x))) + 8] == 1
    for k in range(-2, 14):
        assert O.life_bins([2.0 ** k * T], [5], T)[4 * k + 8] == 1
        assert O.life_bins([2.0 ** k * (1.0 - 1e-12) * T], [5], T)[max(4 * k + 7, 0)] == 1
    assert O.life_bins([1e-9 * T, 0.0, 1e9 * T], [2, 2, 2], T)[[0, 63]].tolist() == [2, 1]
    assert O.life_bins([3.0 * T, 3.0 * T], [1, 0], T).sum() == 0                  # not complexes
    s = O.survival(np.array([1.0, 2.0, 3.0, 4.0, 9.0]), np.array([2, 2, 3, 9, 1]), [0.5, 2.0, 3.5, 10.0])
    assert s.tolist() == [1.0, 0.5, 0.25, 0.0]


def test_thermal_generator_distributions():
    """Reading R18: the thermal-run generator against what the text fixes.  Atom uniform on the
    r0 sphere, Maxwell-Boltzmann velocity with v_r < 0 enforced by negation (so the radial component is half-normal
    and the tangential ones normal); ion position and velocity Gaussian for a harmonic trap of frequency
    q_x Omega / 2^(3/2) at 10 uK -- which is the lowest-order secular frequency (1/2) Omega sqrt(a + q^2/2) at a = 0."""
    from scipy import stats
    n = 40000
    c = I.thermal("Rb87", 3.0, n=n)
    y0, ph, E = O.generate(c.params, c.launch, np.arange(n))
    d = O.derive(c.params)
    kB = 3.1668115634564e-6
    kT_a, kT_i = 3.0e-6 * kB, 10.0e-6 * kB
    r_a, v_a, r_i, v_i = y0[:, 3:6], y0[:, 9:12], y0[:, 0:3], y0[:, 6:9]
    rn = np.linalg.norm(r_a, axis=1)
    assert np.max(np.abs(rn - c.params.r0_a0)) < 1e-9
    nhat = r_a / rn[:, None]
    # uniform on the sphere: cos(theta) uniform on [-1,1], phi uniform on [0, 2 pi)
    assert stats.kstest((nhat[:, 2] + 1) / 2, "uniform").pvalue > 1e-3
    assert stats.kstest(np.mod(np.arctan2(nhat[:, 1], nhat[:, 0]), 2 * np.pi) / (2 * np.pi), "uniform").pvalue > 1e-3
    assert stats.kstest(ph / (2 * np.pi), "uniform").pvalue > 1e-3
    # atom velocity: inward, radial part half-normal, tangential parts normal, all with sigma^2 = k_B T / m_a
    s_a = np.sqrt(kT_a / d["m_a"])
    vr = np.sum(v_a * nhat, axis=1)
    assert vr.max() <= 0.0
    assert stats.kstest(-vr / s_a, "halfnorm").pvalue > 1e-3
    e1 = np.cross(nhat, [0.3, -0.5, 0.8]); e1 /= np.linalg.norm(e1, axis=1)[:, None]
    assert stats.kstest(np.sum(v_a * e1, axis=1) / s_a, "norm").pvalue > 1e-3
    assert abs(E.mean() / kT_a - 1.5) < 4 * np.sqrt(1.5 / n)                       # <E> = 3/2 k_B T
    assert np.allclose(E, 0.5 * d["m_a"] * np.sum(v_a ** 2, axis=1), rtol=1e-14)
    # ion: six independent Gaussians; equipartition <m w^2 x^2> = <m v^2> = k_B T with w = q_x Omega / 2^(3/2)
    s_v = np.sqrt(kT_i / d["m_i"])
    w_h = abs(c.params.q[0]) * d["Omega"] / 2 ** 1.5
    for k in range(3):
        assert stats.kstest(v_i[:, k] / s_v, "norm").pvalue > 1e-3
        assert stats.kstest(r_i[:, k] * w_h / s_v, "norm").pvalue > 1e-3
    assert abs(w_h - 0.5 * d["Omega"] * np.sqrt(0.0 + c.params.q[0] ** 2 / 2)) < 1e-15 * w_h
    assert np.abs(np.corrcoef(np.concatenate([r_i, v_i], axis=1).T) - np.eye(6)).max() < 5 / np.sqrt(n)
    # counter-based: index and first_index commute, different cells differ
    from dataclasses import replace as _r
    y1, _, _ = O.generate(c.params, _r(c.launch, first_index=100), np.arange(5))
    assert np.array_equal(y1, y0[100:105])
    y2, _, _ = O.generate(c.params, _r(c.launch, cell=c.launch.cell + 1), np.arange(5))
    assert not np.array_equal(y2, y0[:5])


def test_exit_localisation_lands_on_the_sphere_inside_the_detecting_step():
    """Reading R7 (amended): for trajectories that were inside the r0 sphere, the recorded exit lies on the sphere to
    1e-13 r0^2 in |d|^2, later than the last accepted state, after fewer than 60 localisation steps -- on a stress
    ensemble with a hot, far-swinging ion and loose tolerances (large steps, oblique crossings of |d| = r0)."""
    from dataclasses import replace as _r
    c = I.thermal("Li7", 100.0, n=400)
    p = _r(c.params, rtol=1e-5, atol=1e-7, t_max_rf=200.0)
    L = _r(c.launch, T_ion_uK=300.0)
    y0, ph, _ = O.generate(p, L, np.arange(400))
    checked = 0
    for k in range(400):
        out, path = O.run(p, y0[k], ph[k], path_cap=100000)
        if out["status"] != 0:
            continue
        dd = np.linalg.norm(path[:, 4:7] - path[:, 1:4], axis=1)
        if not (dd[:-1] < p.r0_a0).any():
            continue                      # started outside and never came in: the exit is the first outward step
        checked += 1
        assert abs(dd[-1] ** 2 - p.r0_a0 ** 2) <= 2e-13 * p.r0_a0 ** 2
        assert path[-2, 0] < out["t_dwell"] and out["n_loc"] < 60
    assert checked > 100
