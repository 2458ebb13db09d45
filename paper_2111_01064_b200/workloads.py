"""Seeded synthetic workloads (BASELINE.json `configs` 0-4; recipe in DESIGN.md §4).

This module is the ONE piece shared by the CPU oracle (`oracle/`) and the CUDA path
(`paper_2111_01064_b200.binding`).  It holds no part of the method: no spline, no waveform,
no inner product.  It only draws parameters, frequency grids, the analytic noise PSD
(an input of the library: it enters through the weights W_k) and noise realisations.

Whatever needs a template (the injected data stream d = h_inj + n, the luminosity scale that
sets SNR = 500, the heterodyne reference h0) is completed by the *consumer* with its own
implementation: tests use `oracle/`, `bench.py` uses the CUDA library.  See `Workload.finish_*`.

Stand-in for: the LDC-1A dataset of PAPER.md:41 (§II) / Fig. 1, which is not available offline.
Shapes follow it: one MBHB, A/E channels, dt=10 s-class rfft grid, SNR of a few hundred.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np

GMSUN_S = 4.925490947e-6          # G M_sun / c^3 in seconds (SURVEY.md §8(c) stand-in)
SEED_BASE = 211101064             # seed = SEED_BASE + config index
F_LO, F_HI = 1.0e-4, 0.05         # analysed band, BASELINE.json configs
SNR_TARGET = 500.0
KAPPA = 0.5                       # taper width, reading (c)9

# (l, m) of BASELINE.json config 3; config 0/1/2/4 use the first entry only.
HM_MODES = ((2, 2), (2, 1), (3, 3), (3, 2), (4, 4), (4, 3))


def psd_sn(f: np.ndarray) -> np.ndarray:
    """Analytic PSD of BASELINE.json config 0 (stand-in for SciRDv1)."""
    f = np.asarray(f, dtype=np.float64)
    s_oms = (15e-12) ** 2
    s_acc = (3e-15) ** 2 / (2.0 * np.pi * f) ** 4
    return s_oms + s_acc * (1.0 + (0.4e-3 / f) ** 2) * (1.0 + (f / 8e-3) ** 4)


def psd_sn_T(f: np.ndarray) -> np.ndarray:
    """Analytic PSD of the T channel for the three-channel variants (Eq. 3 sums over A, E and T; "A=E identical, T
    different").  A stand-in like psd_sn (the paper's SciRDv1 curves are not in PAPER.md): twice the
    optical-metrology floor and a tenth of the acceleration noise, so its shape differs from psd_sn at both ends."""
    f = np.asarray(f, dtype=np.float64)
    s_oms = (15e-12) ** 2
    s_acc = (3e-15) ** 2 / (2.0 * np.pi * f) ** 4
    return 2.0 * s_oms + 0.1 * s_acc * (1.0 + (0.4e-3 / f) ** 2)


def channel_psds(f: np.ndarray, n_c: int) -> np.ndarray:
    """[n_c][n_f]: channels 0, 1 (A, E) share psd_sn, channel 2 (T) has psd_sn_T"""
    return np.stack([psd_sn(f) if c < 2 else psd_sn_T(f) for c in range(n_c)])


@dataclasses.dataclass
class Grid:
    """rfft grid f_k = k*df, k = k_min .. k_min+n_f-1 (reading (c)3)."""
    t_obs: float
    df: float
    k_min: int
    n_f: int

    @property
    def k_max(self) -> int:
        return self.k_min + self.n_f - 1

    def freqs(self) -> np.ndarray:
        return np.arange(self.k_min, self.k_min + self.n_f, dtype=np.float64) * self.df


def make_grid(t_obs: float) -> Grid:
    df = 1.0 / t_obs
    k_min = int(math.ceil(F_LO * t_obs))
    k_max = int(math.floor(F_HI * t_obs))
    return Grid(t_obs=float(t_obs), df=df, k_min=k_min, n_f=k_max - k_min + 1)


def trapezoid_weights(grid: Grid, rule: str = "trapezoid", n_c: int = 2) -> np.ndarray:
    """W_k = 4 df w_k / S_n(f_k) (Eq. 3 discretised; reading (c)4).  n_c = 2: one row [n_f] (A and E share their
    PSD); n_c = 3: one row per channel [3][n_f], the T channel with its own PSD."""
    w = np.ones(grid.n_f)
    if rule == "trapezoid":
        w[0] = 0.5
        w[-1] = 0.5
    if n_c == 2:
        return 4.0 * grid.df * w / psd_sn(grid.freqs())
    return np.ascontiguousarray(4.0 * grid.df * w[None, :] / channel_psds(grid.freqs(), n_c))


def geomspace_exact(lo: float, hi: float, n: int) -> np.ndarray:
    x = np.geomspace(lo, hi, n)
    x[0], x[-1] = lo, hi
    return np.ascontiguousarray(x, dtype=np.float64)


def f_isco_of(mc_s: float, q: float) -> float:
    """Recipe constant used only to PLACE het edges (reading (c)12); the library and the oracle
    each have their own copy inside their stand-in waveform."""
    eta = q / (1.0 + q) ** 2
    m_tot = mc_s * eta ** (-0.6)
    return 6.0 ** (-1.5) / (math.pi * m_tot)


@dataclasses.dataclass
class Workload:
    index: int
    name: str
    path: str                       # "full" | "het"
    grid: Grid
    n_w: int
    n_m: int
    n_c: int
    modes_l: np.ndarray             # int32 [n_m]
    modes_m: np.ndarray             # int32 [n_m]
    c_lm: np.ndarray                # f64 [n_m]
    kappa: float
    params: np.ndarray              # f64 [n_w][P], P = 5 + 2 n_c n_m; 1/D column relative to D_inj until finished
    inj: np.ndarray                 # f64 [P] injection row (1/D = 1 until finished)
    W: np.ndarray                   # f64 [n_f] (n_c = 2) or [n_c][n_f] (n_c = 3: per-channel PSDs)
    noise: Optional[np.ndarray]     # f64 [n_c][n_f][2] or None (noiseless)
    f_nodes: Optional[np.ndarray] = None    # full path
    f_edges: Optional[np.ndarray] = None    # het path
    n_temps: int = 1
    finished: bool = False

    @property
    def P(self) -> int:
        return 5 + 2 * self.n_c * self.n_m

    def finish_distance(self, hh_unit: float) -> None:
        """Second stage of the recipe (reading (c)18): the consumer computes <h|h> of `inj` (which carries
        1/D = 1) with ITS OWN path; D_inj = sqrt(hh)/500, and every 1/D column is rescaled by 1/D_inj."""
        assert not self.finished
        inv_d_inj = SNR_TARGET / math.sqrt(hh_unit)
        self.params[:, 4] *= inv_d_inj
        self.inj[4] *= inv_d_inj
        self.finished = True

    def make_data(self, h_inj: np.ndarray) -> np.ndarray:
        """d = h_inj (+ n); h_inj [n_c][n_f][2] comes from the consumer's own template path."""
        d = np.array(h_inj, dtype=np.float64, copy=True)
        if self.noise is not None:
            d += self.noise
        return d


def _draw_prior(rng: np.random.Generator, n: int, grid: Grid, n_m: int, n_c: int) -> np.ndarray:
    """Prior draws of BASELINE.json config 0: Mc log-U[1e5,1e6] Msun, q U[0.1,1], t_c U[0.5,0.9] T_obs,
    phi_c U[0,2pi), unit-modulus sky factors; 1/D column = u ~ U[0.5,2] (u=1 for row 0), reading (c)18."""
    P = 5 + 2 * n_c * n_m
    p = np.empty((n, P))
    p[:, 0] = GMSUN_S * 10.0 ** rng.uniform(5.0, 6.0, n)
    p[:, 1] = rng.uniform(0.1, 1.0, n)
    p[:, 2] = rng.uniform(0.5, 0.9, n) * grid.t_obs
    p[:, 3] = rng.uniform(0.0, 2.0 * np.pi, n)
    p[:, 4] = rng.uniform(0.5, 2.0, n)
    ang = rng.uniform(0.0, 2.0 * np.pi, (n, n_m * n_c))
    p[:, 5::2] = np.cos(ang)
    p[:, 6::2] = np.sin(ang)
    p[0, 4] = 1.0
    return p


def _draw_ball(rng: np.random.Generator, n: int, inj: np.ndarray, frac: float) -> np.ndarray:
    """Gaussian ball around the injection (reading (c)20)."""
    P = inj.shape[0]
    p = np.tile(inj, (n, 1))
    p[:, 0] *= 1.0 + frac * rng.standard_normal(n)
    p[:, 1] = np.minimum(p[:, 1] * (1.0 + frac * rng.standard_normal(n)), 1.0)
    p[:, 2] += 10.0 * rng.standard_normal(n)
    p[:, 3] += 0.1 * rng.standard_normal(n)
    p[:, 4] *= 1.0 + frac * rng.standard_normal(n)
    n_t = (P - 5) // 2
    delta = 0.05 * rng.standard_normal((n, n_t))
    re, im = p[:, 5::2].copy(), p[:, 6::2].copy()
    p[:, 5::2] = re * np.cos(delta) - im * np.sin(delta)
    p[:, 6::2] = re * np.sin(delta) + im * np.cos(delta)
    return p


def _draw_noise(seed: int, grid: Grid, n_c: int) -> np.ndarray:
    """Re, Im of n_k ~ N(0, S_n(f_k)/(4 df)) (reading (c)16)."""
    rng = np.random.default_rng([seed, 1])
    sigma = np.sqrt(channel_psds(grid.freqs(), n_c) / (4.0 * grid.df))
    n = rng.standard_normal((n_c, grid.n_f, 2))
    n *= sigma[:, :, None]
    return n


_SPEC = {
    #    path    t_obs        n_w     n_m n_nodes/n_bins noise  ball    temps
    0: ("full", 2.0 ** 17,    64,     1,  256,           False, None,   1),
    1: ("het",  2.0 ** 22,    4096,   1,  128,           True,  1e-3,   1),
    2: ("full", 31557600.0,   16384,  1,  1024,          True,  None,   1),
    3: ("het",  2.0 ** 22,    32768,  6,  256,           True,  1e-3,   1),
    4: ("het",  2.0 ** 22,    131072, 1,  512,           True,  1e-2,   16),
}
_NAMES = {0: "cfg0_full_tiny", 1: "cfg1_het", 2: "cfg2_full_search", 3: "cfg3_het_hm", 4: "cfg4_het_mcmc"}


def make_workload(index: int, n_w: Optional[int] = None, t_obs: Optional[float] = None,
                  n_knots: Optional[int] = None, seed_offset: int = 0,
                  noisy: Optional[bool] = None, n_c: int = 2) -> Workload:
    """Build config `index`; the keyword overrides give scaled-down / ragged variants for tests and
    rank-specific draws (seed_offset) for multi-GPU weak scaling.  n_c = 3: the three-channel variant of the
    config (A, E, T with per-channel weights; its own draws, since a parameter row is longer)."""
    path, t0, nw0, n_m, nk0, noisy0, ball, n_temps = _SPEC[index]
    t_obs = t0 if t_obs is None else float(t_obs)
    n_w = nw0 if n_w is None else int(n_w)
    n_knots = nk0 if n_knots is None else int(n_knots)
    noisy = noisy0 if noisy is None else bool(noisy)
    assert n_c in (2, 3)
    seed = SEED_BASE + index + 1000 * seed_offset
    grid = make_grid(t_obs)
    rng = np.random.default_rng(seed)
    l = np.array([lm[0] for lm in HM_MODES[:n_m]], dtype=np.int32)
    m = np.array([lm[1] for lm in HM_MODES[:n_m]], dtype=np.int32)
    c_lm = np.ones(n_m)
    if n_m > 1:
        c_lm[1:] = rng.uniform(0.05, 0.5, n_m - 1)

    # injection = first prior draw of the seeded stream (reading (c)19)
    first = _draw_prior(rng, max(n_w, 1) if ball is None else 1, grid, n_m, n_c)
    inj = first[0].copy()
    if ball is None:
        params = first[:n_w]
    else:
        params = _draw_ball(rng, n_w, inj, ball)
    wl = Workload(index=index, name=_NAMES[index], path=path, grid=grid, n_w=n_w, n_m=n_m, n_c=n_c,
                  modes_l=l, modes_m=m, c_lm=c_lm, kappa=KAPPA,
                  params=np.ascontiguousarray(params), inj=inj,
                  W=trapezoid_weights(grid, n_c=n_c), noise=_draw_noise(seed, grid, n_c) if noisy else None,
                  n_temps=n_temps)
    f_kmin, f_kmax = grid.k_min * grid.df, grid.k_max * grid.df
    if path == "full":
        wl.f_nodes = geomspace_exact(F_LO, F_HI, n_knots)       # reading (c)21
    else:
        f_top = min(f_kmax, f_isco_of(inj[0], inj[1]))           # reading (c)12
        wl.f_edges = geomspace_exact(f_kmin, f_top, n_knots + 1)  # reading (c)11: n_e = n_b + 1
    return wl


def shard_slices(n_items: int, world_size: int) -> list[slice]:
    """Contiguous walker shards for multi-GPU runs (walkers are independent)."""
    base, rem = divmod(n_items, world_size)
    out, lo = [], 0
    for r in range(world_size):
        hi = lo + base + (1 if r < rem else 0)
        out.append(slice(lo, hi))
        lo = hi
    return out
