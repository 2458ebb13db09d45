"""CPU oracle, part 3 — TEST INFRASTRUCTURE ONLY (never imported by the product path; imports nothing of it).

One iteration of the sampler the paper wraps around the likelihood, written out step by step with numpy:

  "This sampler is based on the overall structure of emcee [72] with the parallel tempering scheme from ptemcee
   [73] ... The first is the typical 'stretch' proposal described in [74]"
  stopping tests: extracted SNR <d|h>/sqrt(<h|h>) against a limit, every 150 iterations
                  maximum log L unchanged (within 1) for 30 consecutive checks

The paper gives no formulas for these (they are in its refs [72]-[74]); the readings taken (R25-R28):

  R25 stretch move (Goodman & Weare, the paper's [74], as emcee applies it): the ensemble of one temperature is
      split into two halves; every walker k of the half being updated draws a partner j uniformly from the OTHER
      half and z from g(z) ~ 1/sqrt(z) on [1/a, a] (a = 2) by z = ((a-1) u + 1)^2 / a; proposal
      Y = X_j + z (X_k - X_j); accepted when  ln u' < (d-1) ln z + beta (ln L(Y) - ln L(X_k))  and Y is inside the
      prior box (all priors uniform, Table I); d = number of sampled dimensions.
  R26 tempering (ptemcee): temperature t samples L^beta_t; the move above runs inside each temperature.
  R27 temperature swaps: for t = n_temps-1 down to 1, walker i of temperature t and walker i of temperature t-1
      exchange positions when  ln u < (beta_t - beta_{t-1}) (ln L_{t-1,i} - ln L_{t,i})  (ptemcee pairs the walkers
      through random permutations; the pairing is an input-free identity here: the walkers of a temperature are
      exchangeable).  The sweep is sequential in t, so a walker can climb several rungs in one sweep.
  R28 the random numbers (u_z, u_partner, u_accept, u_swap in [0,1)) are inputs of the step.

Pins (tests/test_oracle_pins.py): z = ((a-1)u+1)^2/a against the closed-form inverse CDF of g; a d-dimensional
Gaussian target keeps its mean and covariance under the move at beta = 1 and is widened by 1/beta at beta < 1
(fails if z^(d-1) is dropped or has the wrong power); swaps always happen at equal betas and follow the textbook
probability on a two-state example; frozen coordinates stay frozen.
"""
from __future__ import annotations

import numpy as np


def stretch_z(u, a=2.0):
    """R25: z with density ~ 1/sqrt(z) on [1/a, a] from u ~ U[0,1)"""
    t = (a - 1.0) * np.asarray(u, dtype=np.float64) + 1.0
    return t * t / a


def stretch_half(x, logL, half, betas, lo, hi, n_dim, a, u_z, u_partner, u_accept, loglike):
    """Update half `half` (0: walkers [0, n/2), 1: walkers [n/2, n)) of every temperature in place.
    x [n_t][n_w][P], logL [n_t][n_w]; u_* [n_t][n_w/2]; loglike(rows [m][P]) -> (logL [m], extra dict of [m] arrays).
    Returns (accepted [n_t][n_w/2] bool, proposals [n_t][n_w/2][P], logL of proposals, extra)."""
    n_t, n_w, P = x.shape
    nh = n_w // 2
    k0, j0 = (0, nh) if half == 0 else (nh, 0)
    z = stretch_z(u_z, a)
    j = np.minimum((np.asarray(u_partner) * nh).astype(np.int64), nh - 1)
    y = np.empty((n_t, nh, P))
    for t in range(n_t):
        for k in range(nh):
            xk, xj = x[t, k0 + k], x[t, j0 + j[t, k]]
            y[t, k] = xj + z[t, k] * (xk - xj)
    inside = np.all((y >= lo) & (y <= hi), axis=2)
    ly, extra = loglike(y.reshape(-1, P))
    ly = ly.reshape(n_t, nh)
    acc = np.zeros((n_t, nh), dtype=bool)
    for t in range(n_t):
        for k in range(nh):
            if not inside[t, k] or not np.isfinite(ly[t, k]):
                continue
            lnq = (n_dim - 1) * np.log(z[t, k]) + betas[t] * (ly[t, k] - logL[t, k0 + k])
            if np.log(u_accept[t, k]) < lnq:
                acc[t, k] = True
                x[t, k0 + k] = y[t, k]
                logL[t, k0 + k] = ly[t, k]
    return acc, y, ly, extra


def temperature_swaps(x, logL, betas, u_swap):
    """R27, in place.  u_swap [n_t-1][n_w]: row t-1 is used for the pair (t, t-1).  Returns swapped [n_t-1][n_w]."""
    n_t, n_w, _ = x.shape
    done = np.zeros((n_t - 1, n_w), dtype=bool)
    for t in range(n_t - 1, 0, -1):
        for i in range(n_w):
            lnq = (betas[t] - betas[t - 1]) * (logL[t - 1, i] - logL[t, i])
            if np.log(u_swap[t - 1, i]) < lnq:
                x[[t, t - 1], i] = x[[t - 1, t], i]
                logL[[t, t - 1], i] = logL[[t - 1, t], i]
                done[t - 1, i] = True
    return done


def population_stats(logL, d_h, h_h):
    """the quantities the two stopping tests look at -> (max log L, its index, max extracted SNR)"""
    logL, d_h, h_h = (np.asarray(v, dtype=np.float64).ravel() for v in (logL, d_h, h_h))
    best, bi = -np.inf, -1
    for i, v in enumerate(logL):
        if np.isfinite(v) and (bi < 0 or v > best):
            best, bi = float(v), i
    snr = -np.inf
    for a, b in zip(d_h, h_h):
        if b > 0 and np.isfinite(a):
            snr = max(snr, a / np.sqrt(b))
    return best, bi, snr


class StopSNR:
    """Module-1 stopping function: stop once the extracted SNR reaches the limit."""

    def __init__(self, limit):
        self.limit = limit

    def check(self, snr):
        return snr >= self.limit


class StopConverged:
    """Module-2 stopping function: stop when the maximum log L has not changed by `tol` (= 1)
    during `n_checks` (= 30) consecutive checks."""

    def __init__(self, n_checks=30, tol=1.0):
        self.n_checks, self.tol, self.ref, self.count = n_checks, tol, None, 0

    def check(self, max_logL):
        if self.ref is None or abs(max_logL - self.ref) >= self.tol:
            self.ref, self.count = max_logL, 0
        else:
            self.count += 1
        return self.count >= self.n_checks


# ------------------------------------------------------------------ counter-based uniforms and a whole run
# R31: when the sampler runs by itself for many iterations (ll_pt_run_het) the uniforms come from a
# counter-based generator that this oracle and the CUDA path each implement: SplitMix64 (Steele, Lea & Flood 2014).
#   mix(z): z ^= z >> 30; z *= 0xBF58476D1CE4E5B9; z ^= z >> 27; z *= 0x94D049BB133111EB; z ^= z >> 31
#   stream key   k = mix(seed + G (8 iter + kind + 1)),  G = 0x9E3779B97F4A7C15
#   r(index)     = mix(k + G (index + 1))        (= the (index+1)-th output of SplitMix64 seeded with k)
#   u            = (r >> 11) 2^-53  in [0, 1)
# kinds: 0, 1, 2 = u_z, u_partner, u_accept of half 0; 3, 4, 5 = the same of half 1; 6 = u_swap.
_G = 0x9E3779B97F4A7C15
_M64 = (1 << 64) - 1


def _mix(z: int) -> int:
    z &= _M64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
    return z ^ (z >> 31)


def stream_key(seed: int, it: int, kind: int) -> int:
    return _mix(seed + _G * (8 * it + kind + 1))


def uniforms(seed: int, it: int, kind: int, n: int) -> np.ndarray:
    k = stream_key(seed, it, kind)
    return np.array([(_mix(k + _G * (i + 1)) >> 11) * 2.0 ** -53 for i in range(n)])


def run(x, logL, betas, lo, hi, n_dim, a, seed, iter0, n_iter, loglike):
    """n_iter iterations (half 0, half 1, swap sweep) in place; returns accepted proposals per temperature."""
    n_t, n_w, _ = x.shape
    nh = n_w // 2
    n_acc = np.zeros(n_t, dtype=np.int64)
    for it in range(iter0, iter0 + n_iter):
        for half in (0, 1):
            u = [uniforms(seed, it, 3 * half + q, n_t * nh).reshape(n_t, nh) for q in range(3)]
            acc, _, _, _ = stretch_half(x, logL, half, betas, lo, hi, n_dim, a, u[0], u[1], u[2], loglike)
            n_acc += acc.sum(axis=1)
        if n_t > 1:
            temperature_swaps(x, logL, betas, uniforms(seed, it, 6, (n_t - 1) * n_w).reshape(n_t - 1, n_w))
    return n_acc
