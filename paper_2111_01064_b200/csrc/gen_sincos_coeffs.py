"""Generator of the sin/cos polynomial coefficients pasted into ll_device.cuh (kernel side only; the oracle
uses libm's sinl/cosl and shares nothing with this file).

sin(pi r/2) = r * S(r^2),  cos(pi r/2) = C(r^2),  |r| <= 1/2 (quarter cycles).  S and C are interpolated at
the Chebyshev nodes of u = r^2 in [0, 1/4] (near-minimax), solved in 60-digit arithmetic, then rounded to the
target type.  Prints hex literals and the maximum error of the rounded polynomial on a 4001-point grid.

    python gen_sincos_coeffs.py
"""
import mpmath as mp
import numpy as np

mp.mp.dps = 60
A, B = mp.mpf(0), mp.mpf(1) / 4


def S(u):
    if u == 0:
        return mp.pi / 2
    r = mp.sqrt(u)
    return mp.sin(mp.pi * r / 2) / r


def C(u):
    return mp.cos(mp.pi * mp.sqrt(u) / 2)


def cheb_fit(F, n):
    global A, B
    xs = [(A + B) / 2 + (B - A) / 2 * mp.cos(mp.pi * (2 * k + 1) / (2 * (n + 1))) for k in range(n + 1)]
    M = mp.matrix(n + 1, n + 1)
    y = mp.matrix(n + 1, 1)
    for i, x in enumerate(xs):
        for j in range(n + 1):
            M[i, j] = x ** j
        y[i] = F(x)
    c = mp.lu_solve(M, y)
    return [c[i] for i in range(n + 1)]


def max_err(F, coeffs, weight):
    e = mp.mpf(0)
    for k in range(4001):
        u = A + (B - A) * mp.mpf(k) / 4000
        p = sum(mp.mpf(ci) * u ** i for i, ci in enumerate(coeffs))
        e = max(e, abs((p - F(u)) * weight(u)))
    return e


def emit(name, F, n, dtype, weight):
    c = cheb_fit(F, n)
    if dtype == "f64":
        r = [float(x) for x in c]
        lits = [float.hex(x) for x in r]
    else:
        r = [float(np.float32(float(x))) for x in c]
        lits = [float.hex(x) + "f" for x in r]
    print(f"// {name}: {n + 1} coefficients ({dtype}), low order first; max |error| {mp.nstr(max_err(F, r, weight), 3)}")
    print("    " + ", ".join(lits))


# FP32-accumulate variant (reading R15): argument in radians, |x| <= pi/4, leading terms exact in binary
# (sin x = x + x^3 S1(x^2), cos x = 1 - x^2/2 + x^4 C2(x^2)) so that no coefficient rounding is coherent at
# the 1e-8 level.
def S1(u):
    if u == 0:
        return -mp.mpf(1) / 6
    x = mp.sqrt(u)
    return (mp.sin(x) / x - 1) / u


def C2(u):
    if u == 0:
        return mp.mpf(1) / 24
    return (mp.cos(mp.sqrt(u)) - 1 + u / 2) / (u * u)


def emit_f32_sequential(name, F, n, weight):
    """float-aware fit: weighted least squares on 200 Chebyshev points; round the lowest free coefficient to
    binary32, freeze it, refit the remaining ones to what is left, repeat"""
    us = [(A + B) / 2 + (B - A) / 2 * mp.cos(mp.pi * (2 * k + 1) / 400) for k in range(200)]
    fs = [F(u) for u in us]
    ws = [weight(u) for u in us]
    fixed = []
    for k in range(n + 1):
        free = list(range(k, n + 1))
        M = mp.matrix(len(us), len(free))
        y = mp.matrix(len(us), 1)
        for i, u in enumerate(us):
            for jj, pw in enumerate(free):
                M[i, jj] = ws[i] * u ** pw
            y[i] = ws[i] * (fs[i] - sum(c * u ** q for q, c in enumerate(fixed)))
        c = mp.lu_solve(M.T * M, M.T * y)
        fixed.append(mp.mpf(float(np.float32(float(c[0])))))
    out = [float(x) for x in fixed]
    print(f"// {name}: {n + 1} coefficients (f32, sequentially rounded), low order first; "
          f"max |error| {mp.nstr(max_err(F, out, weight), 3)}")
    print("    " + ", ".join(float.hex(x) + "f" for x in out))


if __name__ == "__main__":
    emit("S (sin(pi r/2)/r), error weighted by r", S, 5, "f64", lambda u: mp.sqrt(u))
    emit("C (cos(pi r/2))", C, 5, "f64", lambda u: 1)
    B = (mp.pi / 4) ** 2
    emit_f32_sequential("S1 (sin x = x + x^3 S1(x^2)), error weighted by x^3", S1, 3, lambda u: mp.sqrt(u) ** 3)
    emit_f32_sequential("C2 (cos x = 1 - x^2/2 + x^4 C2(x^2)), error weighted by x^4", C2, 2, lambda u: u * u)
    emit_f32_sequential("C2, 4 coefficients", C2, 3, lambda u: u * u)
