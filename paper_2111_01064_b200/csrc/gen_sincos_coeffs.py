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


if __name__ == "__main__":
    emit("S (sin(pi r/2)/r), error weighted by r", S, 6, "f64", lambda u: mp.sqrt(u))
    emit("C (cos(pi r/2))", C, 6, "f64", lambda u: 1)
    emit("S32", S, 4, "f32", lambda u: mp.sqrt(u))
    emit("C32", C, 4, "f32", lambda u: 1)
