"""Where the IA_COS_C0..C8 literals of ia_dev.cuh come from: Remez exchange (absolute error, 60-digit arithmetic,
mpmath) for a polynomial in z = r^2 approximating cos(r) on |r| <= 1.0001 pi/2; prints the coefficients rounded to
double and the error before and after rounding.  Not part of the build; tests/test_host_logic.py checks the literals
independently against a 50-digit cosine.

    python paper_2509_15117_b200/csrc/ia_cos_fit.py
"""
import mpmath as mp
mp.mp.dps = 60
def fit(deg, rmax):
    zmax = rmax**2
    f = lambda z: mp.cos(mp.sqrt(z)) if z > 0 else mp.mpf(1)
    # Remez on [0,zmax] for absolute error
    n = deg + 2
    xs = [zmax*(1-mp.cos(mp.pi*k/(n-1)))/2 for k in range(n)]
    for it in range(30):
        A = mp.matrix(n, n); b = mp.matrix(n, 1)
        for i, x in enumerate(xs):
            for j in range(deg+1): A[i, j] = x**j
            A[i, deg+1] = (-1)**i
            b[i] = f(x)
        sol = mp.lu_solve(A, b)
        c = [sol[j] for j in range(deg+1)]
        err = lambda x: f(x) - sum(c[j]*x**j for j in range(deg+1))
        # find extrema by dense sampling
        N = 4000
        pts = [zmax*mp.mpf(k)/N for k in range(N+1)]
        ev = [err(p) for p in pts]
        ext = [0]
        for k in range(1, N):
            if (ev[k]-ev[k-1])*(ev[k+1]-ev[k]) <= 0: ext.append(k)
        ext.append(N)
        # pick n alternating extrema with largest magnitude
        cand = sorted(ext, key=lambda k: -abs(ev[k]))
        sel = sorted(cand[:n])
        if len(sel) < n: break
        newxs = [pts[k] for k in sel]
        if max(abs(a-b_) for a, b_ in zip(newxs, xs)) < zmax*mp.mpf(10)**-12: xs = newxs; break
        xs = newxs
    return c, max(abs(e) for e in ev)
for deg in (8, 9, 10):
    c, e = fit(deg, mp.pi/2*mp.mpf('1.0001'))
    print(deg, mp.nstr(e, 5))
    if deg in (8,9):
        for j in range(deg, -1, -1): print("   %+.20e," % float(c[j]), " // z^%d, exact %s" % (j, mp.nstr(c[j], 25)))
        # error with double-rounded coefficients, evaluated exactly
        cd = [mp.mpf(float(x)) for x in c]
        zmax = (mp.pi/2)**2
        worst = 0
        for k in range(2001):
            z = zmax*k/2000
            p = sum(cd[j]*z**j for j in range(deg+1))
            worst = max(worst, abs(p - (mp.cos(mp.sqrt(z)) if z>0 else 1)))
        print("   rounded-coefficient max abs err", mp.nstr(worst, 5))
