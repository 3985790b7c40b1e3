"""Where the polynomial coefficients in abm_device.cuh come from (documentation; not needed at run time).

    python paper_1104_2499_b200/csrc/fit_coefficients.py

Near-minimax fits by interpolation at Chebyshev nodes, computed with mpmath at 60 digits, rounded to
double; the printed errors are those of the ROUNDED coefficients in exact arithmetic.
  C_COSPI    cos(pi r) as a polynomial in r^2, |r| <= 1/2                (force, fp64: cospi_f64)
  C_LOG1P    (log1p(r)/r - 1)/r, |r| <= 2^-9                             (Box-Muller, fp64: table-driven log)
  C_BMTRIG   (cos d - 1)/d^2 and sin(d)/d in d^2, |d| <= pi/1024         (Box-Muller, fp64: circle table)
"""
import mpmath as mp

mp.mp.dps = 60


def cheb_fit(f, a, b, deg):
    n = deg + 1
    nodes = [(a + b) / 2 + (b - a) / 2 * mp.cos(mp.pi * (2 * k + 1) / (2 * n)) for k in range(n)]
    A, y = mp.matrix(n, n), mp.matrix(n, 1)
    for i, t in enumerate(nodes):
        for j in range(n):
            A[i, j] = t**j
        y[i] = f(t)
    c = mp.lu_solve(A, y)
    return [float(c[j]) for j in range(n)]


def max_err(f, coefs, a, b, weight=lambda t: 1, n=4000):
    worst = mp.mpf(0)
    for i in range(n + 1):
        t = a + (b - a) * mp.mpf(i) / n
        p = mp.mpf(0)
        for c in reversed(coefs):
            p = p * t + mp.mpf(c)
        worst = max(worst, abs(p - f(t)) * weight(t))
    return worst


def show(name, coefs, err, what):
    print(f"{name}: {what} {mp.nstr(err, 3)}")
    print("    " + ", ".join(repr(c) for c in coefs))


if __name__ == "__main__":
    quarter = mp.mpf(1) / 4
    f = lambda t: mp.cos(mp.pi * mp.sqrt(t))
    c = cheb_fit(f, mp.mpf(0), quarter, 7)
    show("C_COSPI", c, max_err(f, c, mp.mpf(0), quarter), "max abs error")

    R = mp.mpf(2)**-9 * (1 + mp.mpf(2)**-10)
    g = lambda r: mp.mpf(-1) / 2 + r / 3 if abs(r) < mp.mpf(10)**-25 else (mp.log1p(r) / r - 1) / r
    c = cheb_fit(g, -R, R, 3)
    # error of log1p(r) = r (1 + r g(r)) relative to log1p(r)
    show("C_LOG1P", c, max_err(g, c, -R, R, lambda r: r * r / abs(mp.log1p(r)) if r != 0 else 0),
         "max error relative to log1p(r)")

    D2 = (mp.pi / 1024)**2 * (1 + mp.mpf(2)**-20)
    fc = lambda t: mp.mpf(-1) / 2 if t == 0 else (mp.cos(mp.sqrt(t)) - 1) / t
    fs = lambda t: mp.mpf(1) if t == 0 else mp.sin(mp.sqrt(t)) / mp.sqrt(t)
    cc = cheb_fit(fc, mp.mpf(0), D2, 1)
    cs = cheb_fit(fs, mp.mpf(0), D2, 1)
    show("C_BMTRIG[0:2] (cos d - 1)/d^2", cc, max_err(fc, cc, mp.mpf(0), D2, lambda t: t), "max abs error of cos d")
    show("C_BMTRIG[2:4] sin(d)/d", cs, max_err(fs, cs, mp.mpf(0), D2, lambda t: mp.sqrt(t)), "max abs error of sin d")
