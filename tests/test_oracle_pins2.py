"""More pins for the CPU oracle (no GPU needed): the parts of oracle/ia_oracle.cpp that tests/test_oracle_pins.py
left unpinned -- Philox and the word -> uniform map, the GRID and PHILOX direction / phase / energy maps, the error
norm and every branch of the step-size law, the collision times -- and the measured round-off floor of the
adaptive path (oracle against itself compiled with fused multiply-adds).

Each test checks the oracle against something other than itself: published known-answer vectors, closed forms
written out as numbers in tests/golden/, exact rational arithmetic on the published tableau, Kolmogorov-Smirnov
tests against the distributions the readings name, a quadrature of the radial motion.
Citations: PAPER.md (arXiv 2509.15117 text) line numbers; readings R1..R19.
"""
import ctypes as C
import math
import os
import subprocess
from dataclasses import replace
from fractions import Fraction as F

import mpmath as mp
import numpy as np
import pytest
from scipy import integrate, optimize, stats

import ia_inputs as I
from oracle import ia_oracle as O

KB = 3.1668115634564e-6
ME_PER_U = 1822.888486283
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def golden_rows(name):
    with open(os.path.join(GOLD, name)) as fh:
        return [ln.split("#")[0].split() for ln in fh if ln.strip() and not ln.startswith("#")]


# --------------------------------------------------------------------------------------------
# generator: Philox4x32-10, the word -> uniform map, GRID and PHILOX maps (readings R1-R3)
# --------------------------------------------------------------------------------------------
def test_philox_known_answer_vectors():
    """tests/golden/philox4x32_10_kat.txt: the published known-answer vectors of Philox4x32-10 (Salmon et al., SC'11),
    bit for bit.  BASELINE.json configs[2..4] fix the generator as Philox(seed, cell, index)."""
    rows = golden_rows("philox4x32_10_kat.txt")
    assert len(rows) == 3
    for r in rows:
        w = [int(x, 16) for x in r]
        out = O.philox4x32_10(w[0:4], w[4:6])
        assert [int(x) for x in out] == w[6:10], r


def test_u53_exact_values():
    """Reading R2: u = (k + 1/2) 2^-53 with k = (w_even >> 5) 2^26 + (w_odd >> 6), the sum rounded to double.
    Expected values from exact integer arithmetic: k + 1/2 is representable below k = 2^52; from there on the tie
    goes to the even neighbour, so the range is (0, 1] -- never 0 (the thermal generator takes log u)."""
    assert O.u53(0, 0) == 2.0 ** -54
    assert O.u53(0xFFFFFFFF, 0xFFFFFFFF) == 1.0                      # k = 2^53 - 1: k + 1/2 ties to 2^53
    assert O.u53(0, 0x40) == 1.5 * 2.0 ** -53                        # k = 1: the odd word is shifted by 6 ...
    assert O.u53(0x20, 0) == (2.0 ** 26 + 0.5) * 2.0 ** -53          # ... the even one by 5, and weighs 2^26
    assert O.u53(0x1F, 0x3F) == 2.0 ** -54                           # the low bits of both words are dropped
    assert O.u53(0x80000000, 0) == 0.5                               # k = 2^52: tie to even, down
    assert O.u53(0x80000000, 0x40) == (2.0 ** 52 + 2.0) * 2.0 ** -53  # k = 2^52 + 1: tie to even, up
    rng = np.random.default_rng(3)
    for we, wo in rng.integers(0, 2 ** 32, (200, 2)):
        k = (int(we) >> 5) * 2 ** 26 + (int(wo) >> 6)
        assert O.u53(we, wo) == float(F(2 * k + 1, 2)) * 2.0 ** -53   # float(Fraction) rounds to nearest even


def _philox_uniforms(seed, cell, gi, block):
    """The four words of Philox(key = seed; counter = (index_lo, index_hi, cell, block)) as two uniforms, with the
    oracle's (KAT-pinned) Philox and exact integer arithmetic for the map (reading R2)."""
    w = O.philox4x32_10([gi & 0xFFFFFFFF, gi >> 32, cell, block], [seed & 0xFFFFFFFF, seed >> 32])
    u = [float(F(2 * ((int(w[2 * j]) >> 5) * 2 ** 26 + (int(w[2 * j + 1]) >> 6)) + 1, 2)) * 2.0 ** -53 for j in range(2)]
    return u


@pytest.mark.parametrize("domain", [0, 1])
def test_philox_map_word_order_and_counter_layout(domain):
    """Reading R2: block 0 -> (u1, u2) = (cos theta, phi), block 1 -> (u3, u4) = (phase, energy); counter words
    (index_lo, index_hi, cell, block), key = seed; octant cos theta = u1, phi = (pi/2) u2; sphere cos theta = 2 u1 - 1,
    phi = 2 pi u2; phase = 2 pi u3; E = E_min (E_max/E_min)^u4; atom at r0 n, velocity -v0 n, ion at rest at the
    origin.  The index carries into counter word 1 and first_index adds to it."""
    p = I.Params()
    d = O.derive(p)
    seed, cell = 0x0123456789ABCDEF, 77
    L = I.Launch(mode=I.MODE_PHILOX, n=10, domain=domain, phase_mode=1, E_min_uK=2.0, E_max_uK=50.0, seed=seed, cell=cell,
                 first_index=2 ** 32 - 3)
    y0, ph, E = O.generate(p, L, np.arange(6))
    for j in range(6):
        gi = 2 ** 32 - 3 + j
        u1, u2 = _philox_uniforms(seed, cell, gi, 0)
        u3, u4 = _philox_uniforms(seed, cell, gi, 1)
        ct = u1 if domain == 0 else 2 * u1 - 1
        phi = (math.pi / 2 if domain == 0 else 2 * math.pi) * u2
        n = np.array([math.sqrt(1 - ct * ct) * math.cos(phi), math.sqrt(1 - ct * ct) * math.sin(phi), ct])
        assert np.allclose(y0[j, 3:6], p.r0_a0 * n, rtol=0, atol=1e-11)
        assert ph[j] == pytest.approx(2 * math.pi * u3, rel=1e-15)
        E_uK = 2.0 * 25.0 ** u4
        assert E[j] == pytest.approx(E_uK * 1e-6 * KB, rel=1e-14)
        v0 = math.sqrt(2 * E[j] / d["m_a"])
        assert np.allclose(y0[j, 9:12], -v0 * n, rtol=0, atol=1e-14 * v0)
        assert np.all(y0[j, 0:3] == 0.0) and np.all(y0[j, 6:9] == 0.0)
    # fixed phase / fixed energy ignore u3, u4
    y1, ph1, E1 = O.generate(p, replace(L, phase_mode=0, phase0=0.25, E_max_uK=2.0), np.arange(3))
    assert np.all(ph1 == 0.25) and np.all(E1 == 2.0e-6 * KB) and np.allclose(y1[:, 3:6], y0[:3, 3:6], rtol=0, atol=1e-11)


@pytest.mark.parametrize("domain", [0, 1])
def test_philox_map_distributions(domain):
    """'Uniformly randomly chosen' directions and rf phases, log-uniform energies (BASELINE.json
    configs[4]): Kolmogorov-Smirnov tests on cos theta, phi, phase and log E over 40 000 draws, and independence."""
    n = 40000
    p = I.Params()
    L = I.Launch(mode=I.MODE_PHILOX, n=n, domain=domain, phase_mode=1, E_min_uK=1.0, E_max_uK=100.0, seed=11, cell=200)
    y0, ph, E = O.generate(p, L, np.arange(n))
    nh = y0[:, 3:6] / p.r0_a0
    assert np.max(np.abs(np.linalg.norm(nh, axis=1) - 1)) < 1e-14
    ct = nh[:, 2]
    phi = np.mod(np.arctan2(nh[:, 1], nh[:, 0]), 2 * np.pi)
    if domain == 0:
        assert ct.min() > 0 and phi.max() < np.pi / 2 and np.all(nh > 0)             # one octant
        u_ct, u_phi = ct, phi / (np.pi / 2)
    else:
        assert ct.min() < -0.99 and phi.max() > 1.9 * np.pi
        u_ct, u_phi = (ct + 1) / 2, phi / (2 * np.pi)
    u_ph = ph / (2 * np.pi)
    u_E = np.log(E / (1e-6 * KB)) / np.log(100.0)
    for u in (u_ct, u_phi, u_ph, u_E):
        assert 0 <= u.min() and u.max() <= 1
        assert stats.kstest(u, "uniform").pvalue > 1e-3
    assert np.abs(np.corrcoef(np.stack([u_ct, u_phi, u_ph, u_E])) - np.eye(4)).max() < 5 / np.sqrt(n)
    # head-on: the atom's velocity points at the ion, with E = m_a v^2 / 2
    va = y0[:, 9:12]
    d = O.derive(p)
    assert np.allclose(0.5 * d["m_a"] * np.sum(va ** 2, axis=1), E, rtol=1e-14)
    assert np.max(np.abs(np.sum(va * nh, axis=1) / np.linalg.norm(va, axis=1) + 1)) < 1e-14


def test_grid_map_closed_forms():
    """tests/golden/grid_angles.txt (reading R1): cell-centred angles at the corners of the index
    range, on a non-square grid (i = index / N_phi, not / N_theta), octant and sphere; the first index varies phi."""
    p = I.config0().params
    d = O.derive(p)
    v0 = math.sqrt(2 * 10e-6 * KB / d["m_a"])
    for dom, nt, nph, idx, th, phi in golden_rows("grid_angles.txt"):
        L = I.Launch(mode=I.MODE_GRID, n=int(nt) * int(nph), n_theta=int(nt), n_phi=int(nph), domain=int(dom),
                     E_min_uK=10.0, E_max_uK=10.0, phase0=0.7)
        y0, ph, E = O.generate(p, L, [int(idx)])
        th, phi = float(th), float(phi)
        n = np.array([math.sin(th) * math.cos(phi), math.sin(th) * math.sin(phi), math.cos(th)])
        assert np.allclose(y0[0, 3:6], p.r0_a0 * n, rtol=0, atol=2e-12 * p.r0_a0), (dom, nt, nph, idx)
        assert np.allclose(y0[0, 9:12], -v0 * n, rtol=0, atol=2e-12 * v0)
        assert ph[0] == 0.7 and E[0] == pytest.approx(10e-6 * KB, rel=1e-15)
        assert np.all(y0[0, 0:3] == 0.0) and np.all(y0[0, 6:9] == 0.0)
    # consecutive indices walk along phi at fixed theta; a step of N_phi changes theta only
    L = I.config0().launch
    y0, _, _ = O.generate(p, L, [0, 1, 32])
    assert y0[1, 5] == y0[0, 5] and y0[1, 4] > y0[0, 4]             # same cos theta, larger phi
    assert y0[2, 5] < y0[0, 5]                                       # next theta row: smaller cos theta
    assert math.atan2(y0[2, 4], y0[2, 3]) == pytest.approx(math.atan2(y0[0, 4], y0[0, 3]), rel=1e-14)
    # the grid never touches the pole, the symmetry planes or the phi = pi/4 saddle line
    y_all, _, _ = O.generate(p, L, np.arange(L.n))
    assert np.all(y_all[:, 3:6] > 0) and np.min(np.abs(y_all[:, 3] - y_all[:, 4])) > 1.0


# --------------------------------------------------------------------------------------------
# error norm and step-size law of ref [23], reading R5, on a problem with a closed-form step
# --------------------------------------------------------------------------------------------
def controller_constants():
    return {k: mp.mpf(v) for k, v in golden_rows("ode45_controller.txt")}


def test_err_norm_is_the_mixed_max_norm():
    """err = max_i |e_i| / max(|y_i|, |ynew_i|, atol/rtol): hand-made vectors whose maximum sits at a known
    component, through each of the three denominators.  (An RMS norm, a norm on |y| alone or on atol + rtol |y|
    gives other numbers.)"""
    p = replace(I.Params(), rtol=1e-6, atol=1e-8)                   # thr = 1e-2
    y, yn, e = np.zeros(12), np.zeros(12), np.zeros(12)
    y[0], yn[0], e[0] = 2.0, -4.0, 1e-3                              # |ynew| decides: 2.5e-4
    y[5], yn[5], e[5] = 8.0, 1.0, -1.6e-3                            # |y| decides: 2.0e-4
    y[9], yn[9], e[9] = 1e-5, -2e-5, 1.5e-6                          # thr decides: 1.5e-4
    assert O.err_norm(p, y, yn, e) == pytest.approx(2.5e-4, rel=1e-15)
    e[0] = 0.0
    assert O.err_norm(p, y, yn, e) == pytest.approx(2.0e-4, rel=1e-15)
    e[5] = 0.0
    assert O.err_norm(p, y, yn, e) == pytest.approx(1.5e-4, rel=1e-15)
    e[9] = float("nan")
    assert math.isnan(O.err_norm(p, y, yn, e))


# Dormand-Prince 5(4), ref [22], in exact rationals
_A = [[], [F(1, 5)], [F(3, 40), F(9, 40)], [F(44, 45), F(-56, 15), F(32, 9)],
      [F(19372, 6561), F(-25360, 2187), F(64448, 6561), F(-212, 729)],
      [F(9017, 3168), F(-355, 33), F(46732, 5247), F(49, 176), F(-5103, 18656)],
      [F(35, 384), F(0), F(500, 1113), F(125, 192), F(-2187, 6784), F(11, 84)]]
_B = [F(35, 384), F(0), F(500, 1113), F(125, 192), F(-2187, 6784), F(11, 84), F(0)]
_BH = [F(5179, 57600), F(0), F(7571, 16695), F(393, 640), F(-92097, 339200), F(187, 2100), F(1, 40)]


def linear_step_polynomials():
    """For y' = M y one explicit RK step is y_new = R(hM) y and the embedded error estimate e = E(hM) y with
    R(z) = 1 + z sum_s b_s P_s(z), E(z) = z sum_s (b_s - bhat_s) P_s(z), P_s(z) = 1 + z sum_l a_sl P_l(z)."""
    def add(a, b):
        return [(a[i] if i < len(a) else 0) + (b[i] if i < len(b) else 0) for i in range(max(len(a), len(b)))]
    P = []
    for s in range(7):
        acc = [F(0)]
        for l, a in enumerate(_A[s]):
            acc = add(acc, [a * c for c in P[l]])
        P.append([F(1)] + acc)
    def comb(w):
        out = [F(0)]
        for s in range(7):
            out = add(out, [F(0)] + [w[s] * c for c in P[s]])
        return (out + [F(0)] * 8)[:8]
    R = comb(_B)
    R[0] = F(1)
    return R, comb([b - bh for b, bh in zip(_B, _BH)])


def test_linear_step_polynomials_are_the_known_ones():
    R, E = linear_step_polynomials()
    assert R == [1, 1, F(1, 2), F(1, 6), F(1, 24), F(1, 120), F(1, 600), 0]      # the DP5 stability polynomial
    assert E == [0, 0, 0, 0, 0, F(-97, 120000), F(13, 40000), F(-1, 24000)]


class LinearIon:
    """Lone ion (alpha = 0: no pair force) in a static trap (q = 0): three uncoupled linear oscillators
    x_k'' = -kappa_k x_k, kappa_k = a_k Omega^2/4 -- kappa < 0 on an anti-trapping axis.
    M^2 = -kappa on each axis, so R(hM) y and E(hM) y are finite sums, evaluated here in 40-digit arithmetic."""

    def __init__(self, a, rtol, atol, h_max_rf=0.25, max_steps=2 ** 31):
        self.p = replace(I.Params(), alpha_au=0.0, r0_a0=1e12, rtol=rtol, atol=atol, a=a, q=(0.0, 0.0, 0.0),
                         t_max_rf=1e4, h_max_rf=h_max_rf, max_steps=max_steps)
        mp.mp.dps = 40
        Om = mp.mpf(self.p.omega_rf_au)
        self.kappa = [mp.mpf(x) * Om * Om / 4 for x in a]
        self.T = 2 * mp.pi / Om
        self.R, self.E = [[mp.mpf(c.numerator) / c.denominator for c in poly] for poly in linear_step_polynomials()]

    def step(self, y, h):
        """y = [(x_k, v_k)] -> (ynew, e)"""
        yn, en = [], []
        for (x, v), kap in zip(y, self.kappa):
            vec, hk = (x, v), mp.mpf(1)
            a, b = [mp.mpf(0)] * 2, [mp.mpf(0)] * 2
            for k in range(8):
                a = [a[0] + self.R[k] * hk * vec[0], a[1] + self.R[k] * hk * vec[1]]
                b = [b[0] + self.E[k] * hk * vec[0], b[1] + self.E[k] * hk * vec[1]]
                vec, hk = (vec[1], -kap * vec[0]), hk * h
            yn.append(tuple(a))
            en.append(tuple(b))
        return yn, en

    def err(self, y, yn, e):
        thr = mp.mpf(self.p.atol) / mp.mpf(self.p.rtol)
        return max(max(abs(ex) / max(abs(x), abs(xn), thr), abs(ev) / max(abs(v), abs(vn), thr))
                   for (x, v), (xn, vn), (ex, ev) in zip(y, yn, e))

    def expected_attempts(self, y0, n_attempts, const):
        """The attempts the controller of tests/golden/ode45_controller.txt makes from y0: a list of
        (accepted, branch, h, err/rtol, t after, state after)."""
        rtol = mp.mpf(self.p.rtol)
        thr = mp.mpf(self.p.atol) / rtol
        h_max, t_max = mp.mpf(self.p.h_max_rf) * self.T, mp.mpf(self.p.t_max_rf) * self.T
        y = [(mp.mpf(float(y0[k])), mp.mpf(float(y0[6 + k]))) for k in range(3)]
        rho = max(max(abs(v) / max(abs(x), thr), abs(kap * x) / max(abs(v), thr)) for (x, v), kap in zip(y, self.kappa))
        rho /= const["safety"] * rtol ** const["order_exponent"]
        h = min(h_max, t_max)
        if h * rho > 1:
            h = 1 / rho
        t, failed, log = mp.mpf(0), False, []
        for _ in range(n_attempts):
            yn, e = self.step(y, h)
            x = self.err(y, yn, e) / rtol
            if x <= 1:
                t, y = t + h, yn
                if failed:
                    branch, hn = "accept-after-reject", h
                else:
                    f = x ** const["order_exponent"] / const["safety"]
                    branch = "grow" if f > 1 / const["growth_max"] else "grow-clamped"
                    hn = h / max(1 / const["growth_max"], f)
                if hn > h_max:
                    branch, hn = branch + "+hmax", h_max
                log.append((True, branch, h, x, t, y))
                failed = False
            else:
                if failed:
                    branch, hn = "halve", h * const["shrink_repeat"]
                else:
                    f = const["safety"] * (1 / x) ** const["order_exponent"]
                    branch = "shrink" if f > const["shrink_min"] else "shrink-clamped"
                    hn = h * max(const["shrink_min"], f)
                log.append((False, branch, h, x, t, y))
                failed = True
            h = hn
        return log

    def y0(self, z0, v0):
        y = np.zeros(12)
        y[0], y[1], y[2], y[6], y[8], y[3] = 0.3 * z0, -2.0 * z0, z0, 0.1 * v0, v0, 1e6
        return y


def test_one_step_and_error_estimate_on_the_linear_problem():
    """oracle_step against R(hM) y and E(hM) y, and oracle_err_norm of that step against the closed form."""
    S = LinearIon((-1.2, 2.0, 4.0), 1e-6, 1e-8)
    y0 = S.y0(10.0, 3e-9)
    for h_rf in (0.25, 0.03, 0.004):
        h = h_rf * float(S.T)
        ynew, e = O.step(S.p, 0.0, 0.0, y0, h)
        y = [(mp.mpf(float(y0[k])), mp.mpf(float(y0[6 + k]))) for k in range(3)]
        yn, en = S.step(y, mp.mpf(h))
        for k in range(3):
            assert ynew[k] == pytest.approx(float(yn[k][0]), rel=1e-13)
            assert ynew[6 + k] == pytest.approx(float(yn[k][1]), rel=1e-13)
            # the estimate is a difference of nearly equal sums: its rounding scales with |h k_l|, not with |e|
            assert e[k] == pytest.approx(float(en[k][0]), abs=4e-16 * abs(float(yn[k][1])) * h + 1e-30)
            assert e[6 + k] == pytest.approx(float(en[k][1]), abs=4e-16 * abs(float(S.kappa[k] * yn[k][0])) * h + 1e-40)
        assert np.all(ynew[3:6] == y0[3:6]) and np.all(e[3:6] == 0) and np.all(e[9:12] == 0)   # the free atom at rest
        assert O.err_norm(S.p, y0, ynew, e) == pytest.approx(float(S.err(y, yn, en)), rel=1e-9 / h_rf ** 2 * 1e-4 + 1e-12)


@pytest.mark.parametrize("a_z,rtol,atol,z0,v0,h_max_rf,n_att,branches", [
    (4.0, 1e-6, 1e-8, 10.0, 0.0, 0.25, 25, ["shrink", "accept-after-reject", "grow"]),
    (400.0, 1e-6, 1e-8, 10.0, 0.0, 0.25, 12, ["shrink-clamped", "halve", "halve", "halve", "accept-after-reject", "grow"]),
    (0.04, 1e-8, 1e-20, 10.0, 3e-9, 0.02, 12, ["grow-clamped", "grow-clamped", "grow-clamped", "grow-clamped+hmax", "grow+hmax"]),
])
def test_step_size_law_branch_by_branch(a_z, rtol, atol, z0, v0, h_max_rf, n_att, branches):
    """The accepted times and states, the accept / reject counts and the first step of the oracle's adaptive run
    against the controller of ref [23] as tests/golden/ode45_controller.txt states it, with the error of every
    attempt from the closed-form step: first-step rule, max-norm, accept test, 0.8 (rtol/err)^(1/5) with the 1/5
    growth and 0.1 shrink limits, halving on repeated rejection, no growth on the accept after a rejection, h_max."""
    const = controller_constants()
    S = LinearIon((-0.3 * a_z, 0.5 * a_z, a_z), rtol, atol, h_max_rf=h_max_rf, max_steps=n_att)
    y0 = S.y0(z0, v0)
    log = S.expected_attempts(y0, n_att, const)
    assert [b for _, b, *_ in log][:len(branches)] == branches
    # no decision of the scenario sits within 5 % of its threshold (round-off cannot flip it)
    assert all(abs(float(x) - 1) > 0.05 for _, _, _, x, _, _ in log)
    out, path = O.run(S.p, y0, path_cap=n_att + 1)
    acc = [l for l in log if l[0]]
    assert out["status"] == 4 and out["steps_acc"] == len(acc) and out["steps_rej"] == n_att - len(acc)
    assert out["h_first"] == pytest.approx(float(log[0][2]), rel=1e-14)
    assert len(path) == len(acc) + 1
    for row, (_, _, h, x, t, y) in zip(path[1:], acc):
        assert row[0] == pytest.approx(float(t), rel=2e-11)          # h inherits err^(1/5): 1e-12 per step
        for k in range(3):
            assert row[1 + k] == pytest.approx(float(y[k][0]), rel=1e-9, abs=1e-9 * z0)
            assert row[7 + k] == pytest.approx(float(y[k][1]), rel=1e-9, abs=1e-9 * z0 * math.sqrt(abs(float(S.kappa[2]))))


# --------------------------------------------------------------------------------------------
# collision times (reading R6)
# --------------------------------------------------------------------------------------------
def turning_time_quadrature(p, E):
    """Head-on, trap off: time from r0 to the inner turning point of the relative motion,
    t = int_{r_min}^{r0} dr / sqrt((2/mu)(E_cm - V(r))), r = r_min + (r0 - r_min) s^2."""
    m_i, m_a = p.m_ion_u * ME_PER_U, p.m_atom_u * ME_PER_U
    mu = m_i * m_a / (m_i + m_a)
    C4 = p.alpha_au / 2
    C8 = C4 ** 2 / (4 * p.De_K * KB)
    V = lambda r: C8 / r ** 8 - C4 / r ** 4
    v0 = math.sqrt(2 * E / m_a)
    r0 = p.r0_a0
    E_cm = 0.5 * mu * v0 ** 2 + V(r0)
    rad = lambda r: (2 / mu) * (E_cm - V(r))
    r_min = optimize.brentq(rad, 10.0, 0.9 * (2 * C8 / C4) ** 0.25, xtol=1e-15, rtol=1e-15)
    f = lambda s: 2 * (r0 - r_min) * s / math.sqrt(max(rad(r_min + (r0 - r_min) * s * s), 1e-300))
    val, _ = integrate.quad(f, 0, 1, epsabs=0, epsrel=1e-13, limit=1000)
    return val, v0


@pytest.mark.parametrize("atom,E_uK", [("Li7", 10.0), ("Rb87", 10.0), ("Rb87", 1.5)])
def test_collision_time_is_the_turning_point(atom, E_uK):
    """R6: the collision time t_n + h s_n / (s_n - s_{n+1}) against the closed-form turning time of the trap-free
    head-on bounce, to a small fraction of the step that straddles it (an interpolation with the wrong end, sign or
    weight is off by a whole step fraction); one bounce: t_first = t_last, t_life = 0."""
    p = replace(I.Params().with_atom(atom), a=(0, 0, 0), q=(0, 0, 0), t_max_rf=1e5)
    t_turn, v0 = turning_time_quadrature(p, E_uK * 1e-6 * KB)
    out, path = O.run(p, I.impact_ic(0.0, p.r0_a0, v0), path_cap=100000)
    assert out["status"] == 0 and out["n_coll"] == 1 and out["n_tp"] == 1
    assert out["t_first"] == out["t_last"] and out["t_life"] == 0.0
    k = int(np.searchsorted(path[:, 0], out["t_first"]))
    h_loc = path[k, 0] - path[k - 1, 0]
    assert path[k - 1, 0] < t_turn < path[k, 0]                      # the quadrature's time lies in that very step
    assert abs(out["t_first"] - t_turn) < 2e-3 * h_loc
    assert abs(out["t_first"] - t_turn) < 1e-9 * t_turn
    assert abs(out["t_dwell"] / 2 - t_turn) < 1e-2 * t_turn          # elastic: out as fast as in, up to the truncation
    # error of the outgoing energy, which the well amplifies by D_e/E (3e-3 at 1.5 uK, reading R15)


def test_first_and_last_collision_times_of_a_complex():
    """R6 on a complex of config 1 (PAPER.md:30 'more than a single bounce'): t_first and t_last against the
    first and last short-range minimum of r(t) read off the accepted states by a parabola through the three
    samples around each minimum of |d|^2 -- another estimator, good to a fraction of the local step."""
    c = I.config1(512)
    T = O.derive(c.params)["T_rf"]
    found = 0
    for idx in I.subgrid_indices(512, 64):
        y0, ph, _ = O.generate(c.params, c.launch, [idx])
        out, path = O.run(c.params, y0[0], ph[0], path_cap=400000)
        if not (2 <= out["n_coll"] <= 40) or out["status"] != 0 or len(path) != out["steps_acc"] + 1:
            continue
        found += 1
        t = path[:-1, 0]                                             # accepted states (the last row is the localised exit)
        d = path[:-1, 4:7] - path[:-1, 1:4]
        r2 = np.sum(d * d, axis=1)
        k = np.where((r2[1:-1] < r2[:-2]) & (r2[1:-1] <= r2[2:]) & (r2[1:-1] < c.params.r_coll_a0 ** 2))[0] + 1
        assert len(k) == out["n_coll"]
        def vertex(j):
            q = np.polyfit(t[j - 1:j + 2] - t[j], r2[j - 1:j + 2], 2)
            return t[j] - q[1] / (2 * q[0])
        for tc, j in ((out["t_first"], k[0]), (out["t_last"], k[-1])):
            h_loc = max(t[j + 1] - t[j], t[j] - t[j - 1])
            assert abs(tc - vertex(j)) < 0.5 * h_loc, (idx, tc / T, vertex(j) / T)
        assert out["t_life"] == out["t_last"] - out["t_first"] > 0
        if found == 4:
            break
    assert found == 4


# --------------------------------------------------------------------------------------------
# round-off floor of the adaptive path (reading R19)
# --------------------------------------------------------------------------------------------
def test_roundoff_floor_of_the_adaptive_path_oracle_against_itself(tmp_path):
    """BASELINE.json north_star asks that final observables of non-chaotic trajectories agree to a relative 1e-8
    between the two implementations.  That is a same-algorithm agreement near the FP64 floor (reading R15): this test
    MEASURES the floor, with nothing but the oracle -- its source compiled a second time with fused multiply-adds
    (-ffp-contract=fast -mfma), i.e. the same algorithm with different rounding -- on all 1 024 trajectories of
    config 0.  Every step sequence is identical; t_dwell and the exit velocity agree to < 1e-8; ke_ion, which
    carries the micromotion phase 2 pi t/T_rf, does not: its maximum over the grid is 4e-8 (median 1.2e-9).
    DESIGN.md reading R19 records the table; tests/test_gpu_parity.py holds the CUDA path to twice these numbers."""
    if "fma" not in open("/proc/cpuinfo").read():
        pytest.skip("host CPU has no FMA units: the second build would be the same program")
    lib = tmp_path / "libia_oracle_fma.so"
    src = os.path.join(os.path.dirname(O.__file__), "ia_oracle.cpp")
    flags = [f for f in O.CXXFLAGS if f != "-ffp-contract=off"] + ["-ffp-contract=fast", "-mfma"]
    subprocess.run(["g++", *flags, "-o", str(lib), src], check=True)
    L = C.CDLL(str(lib))
    L.oracle_run_generated.argtypes = [C.POINTER(O.OracleParams), C.POINTER(O.OracleGen), C.POINTER(C.c_uint64),
                                       C.c_uint64, C.c_uint64, C.c_void_p, C.c_int]
    c = I.config0()
    nthr = os.cpu_count() or 1
    a = O.run_generated(c.params, c.launch, nthreads=nthr)
    b = np.zeros(c.launch.n, dtype=O.OUTCOME_DTYPE)
    assert L.oracle_run_generated(C.byref(O.to_params(c.params)), C.byref(O.to_gen(c.launch)), None, 0, c.launch.n,
                                  b.ctypes.data, nthr) == 0
    assert np.array_equal(a["steps_acc"], b["steps_acc"]) and np.array_equal(a["steps_rej"], b["steps_rej"])
    assert np.array_equal(a["n_coll"], b["n_coll"]) and np.all(a["n_coll"] == 1)
    e_t = np.abs(a["t_dwell"] / b["t_dwell"] - 1)
    e_k = np.abs(a["ke_ion"] / b["ke_ion"] - 1)
    e_v = np.linalg.norm(a["va_f"] - b["va_f"], axis=1) / np.linalg.norm(b["va_f"], axis=1)
    print(f"oracle vs oracle+fma, config 0: t_dwell max {e_t.max():.2e} median {np.median(e_t):.2e}; "
          f"ke_ion max {e_k.max():.2e} median {np.median(e_k):.2e}; va_f max {e_v.max():.2e} median {np.median(e_v):.2e}")
    assert e_t.max() < 2e-9 and e_v.max() < 5e-9                       # below the 1e-8 of north_star
    assert 1e-8 < e_k.max() < 1e-7 and 3e-10 < np.median(e_k) < 3e-9   # the floor of ke_ion is NOT below it


# --------------------------------------------------------------------------------------------
# the oracle under AddressSanitizer and UndefinedBehaviorSanitizer
# --------------------------------------------------------------------------------------------
_ASAN_DRIVER = r"""
#include <cstdio>
#include <cstring>
#include <vector>
#include "ia_oracle.h"
int main() {
    oracle_params p;
    std::memset(&p, 0, sizeof(p));
    p.m_ion_u = 173.94; p.m_atom_u = 86.909; p.alpha_au = 319.2;
    p.a[0] = -0.0005; p.a[1] = -0.0005; p.a[2] = 0.001; p.q[0] = 0.1; p.q[1] = -0.1; p.q[2] = 0.0;
    p.omega_rf_au = 3.0396596921148e-10; p.De_K = 1.0; p.r0_a0 = 5000.0; p.rtol = 1e-10; p.atol = 1e-12;
    p.t_max_rf = 60.0; p.h_max_rf = 0.25; p.r_coll_a0 = 500.0; p.max_steps = 1ull << 31;
    unsigned long long done = 0, complexes = 0;
    for (int mode = 1; mode <= 3; ++mode) {           /* GRID, PHILOX, THERMAL */
        oracle_gen g;
        std::memset(&g, 0, sizeof(g));
        g.mode = mode; g.domain = mode == 1 ? 0 : 1; g.phase_mode = mode == 1 ? 0 : 1; g.n_theta = 7; g.n_phi = 9;
        g.E_min_uK = 1.5; g.E_max_uK = mode == 2 ? 100.0 : 1.5; g.seed = 12345; g.cell = 7; g.first_index = mode == 2 ? (1ull << 33) - 5 : 0;
        g.T_atom_uK = 3.0; g.T_ion_uK = 10.0;
        const uint64_t n = 63;
        std::vector<oracle_outcome> out(n);
        if (oracle_run_generated(&p, &g, nullptr, 0, n, out.data(), 3) != 0) return 2;
        for (const auto &o : out) { ++done; complexes += o.n_coll >= 2; if (o.status < 0 || o.status > 4) return 3; }
    }
    /* trace and path buffers at their exact sizes */
    double y0[12], ph, E;
    oracle_gen g; std::memset(&g, 0, sizeof(g)); g.mode = 1; g.n_theta = 4; g.n_phi = 4; g.E_min_uK = g.E_max_uK = 1.5;
    if (oracle_generate(&p, &g, 5, y0, &ph, &E) != 0) return 4;
    std::vector<double> states(13 * 41);
    oracle_trace(&p, y0, ph, 1e8, 40, states.data());
    std::vector<double> path(13 * 100);
    oracle_outcome o; uint64_t len = 0;
    oracle_run(&p, y0, ph, &o, path.data(), 100, &len);
    if (len > 100) return 5;
    std::printf("%llu trajectories, %llu complexes\n", done, complexes);
    return 0;
}
"""


def test_oracle_is_clean_under_asan_and_ubsan(tmp_path):
    """The oracle's source compiled with -fsanitize=address,undefined (no recovery) into a small driver that runs all
    three generators (ragged counts, an index that carries into the second counter word, three worker threads),
    a fixed-step trace and a path dump into buffers of exactly the documented sizes: exits 0 with no report."""
    import shutil
    if shutil.which("g++") is None:
        pytest.skip("g++ not on PATH")
    odir = os.path.dirname(O.__file__)
    src = tmp_path / "driver.cpp"
    src.write_text(_ASAN_DRIVER)
    exe = tmp_path / "driver"
    flags = ["-std=c++17", "-O1", "-g", "-ffp-contract=off", "-pthread", "-fsanitize=address,undefined",
             "-fno-sanitize-recover=all", "-fno-omit-frame-pointer"]
    r = subprocess.run(["g++", *flags, "-I", odir, "-o", str(exe), str(src), os.path.join(odir, "ia_oracle.cpp")],
                       capture_output=True, text=True)
    if r.returncode != 0 and "asan" in (r.stderr or "").lower():
        pytest.skip("sanitizer runtime not installed")
    assert r.returncode == 0, r.stderr[-2000:]
    run = subprocess.run([str(exe)], capture_output=True, text=True, timeout=300,
                         env={**os.environ, "ASAN_OPTIONS": "detect_leaks=1:abort_on_error=0"})
    assert run.returncode == 0, (run.stdout[-500:], run.stderr[-3000:])
    assert "189 trajectories" in run.stdout and "ERROR" not in run.stderr
