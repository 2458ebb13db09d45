// ll_kernels.cuh — the sm_100a kernels of libll_b200 (steps F0-F4, H0-H3 of DESIGN.md §2).
//
// Device layouts ("sorted position" p = index of a walker after the band-top counting sort; n_wp = n_w
// rounded up to the walker-block size):
//   g4   [n_f_pad][4]   W_i * conj(d^c_i): (A re, A im, E re, E im); im already negated          (F0)
//   Wd   [n_f_pad]      W_i, zero in the padding
//   Y    [n_m*2][n_nodes][n_wp]   node values, sys = 2 m + kind (0 amplitude, 1 phase in quarter cycles)
//   C    [n_nodes-1][n_m][8][n_wp] cubic coefficients per interval: (y, b, c, d) amplitude, then phase
//   TF   [n_m][2][2][n_wp]         transfer factors T^c_m (re, im)
//   part [n_tiles][NQ][n_wp]       per-(frequency tile, walker) partial sums
#pragma once
#include <limits.h>
#include "ll_device.cuh"

namespace ll {

constexpr int kMaxModes = 8;
constexpr int kNC = 2;

// ---------------------------------------------------------------------------------------------------
// F0: pre-weighted data and <d|d>          (Eq. 3; "we transform the data")
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ double block_sum_256(double v, double *sh)
{
    v = warp_sum(v);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) sh[wid] = v;
    __syncthreads();
    double r = 0.0;
    if (wid == 0) {
        r = (lane < (int)(blockDim.x >> 5)) ? sh[lane] : 0.0;
        r = warp_sum(r);
    }
    __syncthreads();
    return r; // valid in warp 0
}

__global__ void __launch_bounds__(256) k_preweight(const double *__restrict__ d, const double *__restrict__ W,
                                                   long long n_f, double *__restrict__ g4,
                                                   double *__restrict__ Wd, double *__restrict__ dd_part)
{
    __shared__ double sh[8];
    double acc = 0.0, comp = 0.0; // Neumaier-compensated per-thread sum
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_f; i += (long long)gridDim.x * blockDim.x) {
        const double w = W[i];
        const double2 a = reinterpret_cast<const double2 *>(d)[i];
        const double2 e = reinterpret_cast<const double2 *>(d)[n_f + i];
        reinterpret_cast<double4 *>(g4)[i] = make_double4(w * a.x, -(w * a.y), w * e.x, -(w * e.y));
        Wd[i] = w;
        const double term = w * (a.x * a.x + a.y * a.y + e.x * e.x + e.y * e.y);
        const double t = acc + term;
        comp += (fabs(acc) >= fabs(term)) ? ((acc - t) + term) : ((term - t) + acc);
        acc = t;
    }
    const double tot = block_sum_256(acc + comp, sh);
    if (threadIdx.x == 0) dd_part[blockIdx.x] = tot;
}

// out[0] = sum of part[0..n) in a fixed order (single block; deterministic)
__global__ void __launch_bounds__(256) k_sum_parts(const double *__restrict__ part, int n, double *__restrict__ out)
{
    __shared__ double sh[8];
    double acc = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) acc += part[i];
    const double tot = block_sum_256(acc, sh);
    if (threadIdx.x == 0) out[0] = tot;
}

// ---------------------------------------------------------------------------------------------------
// Band -> bin range per walker, sort key histogram, active-pair count          (reading R10)
// ---------------------------------------------------------------------------------------------------
struct GridInfo {
    long long k_min;
    long long n_f;
    double df;
};

struct StandinInfo {
    int n_m;
    int m_max;
    int mode_m[kMaxModes];
    double kappa;
};

__device__ __forceinline__ void standin_masses(double Mc, double q, double &Mtot, double &eta, double &f_isco)
{
    eta = q / ((1.0 + q) * (1.0 + q));
    Mtot = Mc * pow(eta, -0.6);
    f_isco = 0x1.16b28f55d72d4p-4 / (kPi * Mtot); // 6^(-3/2) = 0.06804138174397717
}

// bin range [lo, hi) of walker w's band: stand-in parameters (reading R10), a caller band [n_w][2], or the whole grid
__device__ __forceinline__ void band_bins(int use_standin, const double *__restrict__ params, int P,
                                          const double *__restrict__ band, int w, const GridInfo &g, const StandinInfo &si,
                                          long long &lo, long long &hi)
{
    double f_lo, f_hi;
    if (use_standin) {
        double Mtot, eta, fi;
        standin_masses(params[(size_t)w * P], params[(size_t)w * P + 1], Mtot, eta, fi);
        f_lo = bin_freq(g.k_min, 0, g.df);
        const double top = (1.0 + si.kappa) * fi * (0.5 * (double)si.m_max);
        const double f_last = bin_freq(g.k_min, g.n_f - 1, g.df);
        f_hi = (top < f_last) ? top : f_last;
    } else if (band) {
        f_lo = band[2 * (size_t)w];
        f_hi = band[2 * (size_t)w + 1];
    } else {
        f_lo = -INFINITY;
        f_hi = INFINITY;
    }
    lo = first_bin_ge(f_lo, g.k_min, g.n_f, g.df);
    hi = first_bin_gt(f_hi, g.k_min, g.n_f, g.df);
    if (!(f_lo <= f_hi) || hi <= lo) { lo = 0; hi = 0; }
}

__global__ void __launch_bounds__(256)
k_band_prep(int use_standin, const double *__restrict__ params, int P, const double *__restrict__ band, int n_w,
            GridInfo g, StandinInfo si, int key_gran, int *__restrict__ ilo_w, int *__restrict__ ihi_w,
            int *__restrict__ key_w, int *__restrict__ hist, unsigned long long *__restrict__ pairs)
{
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    long long span = 0;
    if (w < n_w) {
        long long lo, hi;
        band_bins(use_standin, params, P, band, w, g, si, lo, hi);
        ilo_w[w] = (int)lo;
        ihi_w[w] = (int)hi;
        const int key = (int)(hi / key_gran);
        key_w[w] = key;
        atomicAdd(&hist[key], 1);
        span = hi - lo;
    }
    // integer atomics: deterministic
    unsigned long long s = (unsigned long long)span;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0 && s) atomicAdd(pairs, s * (unsigned long long)si.n_m);
}

// The same three steps (band -> bin range, sort by band top, scatter) for batches of up to 1024 walkers in ONE
// block (Module-1 sized batches are latency-bound: one launch instead of three plus two memsets).  Rank of a walker
// = number of walkers with a smaller (top bin, index): an O(n^2) count over shared memory, n <= 1024.
__global__ void __launch_bounds__(1024)
k_band_sort_small(int use_standin, const double *__restrict__ params, int P, const double *__restrict__ band, int n_w,
                  int n_wp, GridInfo g, StandinInfo si, int *__restrict__ perm, int *__restrict__ ilo_s,
                  int *__restrict__ ihi_s, unsigned long long *__restrict__ pairs)
{
    __shared__ int s_hi[1024];
    __shared__ unsigned long long s_span[32];
    const int w = threadIdx.x;
    long long lo = 0, hi = 0;
    if (w < n_w) band_bins(use_standin, params, P, band, w, g, si, lo, hi);
    s_hi[w] = (w < n_w) ? (int)hi : INT_MAX;
    unsigned long long s = (unsigned long long)(hi - lo);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((w & 31) == 0) s_span[w >> 5] = s;
    __syncthreads();
    if (w == 0) {
        unsigned long long t = 0;
        for (int k = 0; k < 32; ++k) t += s_span[k];
        pairs[0] = t * (unsigned long long)si.n_m;
    }
    if (w < n_w) {
        const int mine = (int)hi;
        int rank = 0;
        for (int k = 0; k < n_w; ++k) {
            const int other = s_hi[k];
            rank += (other < mine) || (other == mine && k < w);
        }
        perm[rank] = w;
        ilo_s[rank] = (int)lo;
        ihi_s[rank] = (int)hi;
    } else if (w < n_wp) {
        perm[w] = -1;
        ilo_s[w] = 0;
        ihi_s[w] = 0;
    }
}

// exclusive scan of hist[0..n) in place (single block of 1024 threads, n <= 1024*8)
__global__ void __launch_bounds__(1024) k_scan_hist(int *__restrict__ hist, int n)
{
    __shared__ int wsum[32];
    const int per = (n + 1023) / 1024;
    const int b = threadIdx.x * per;
    int loc[8];
    int s = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        loc[k] = 0;
        if (k < per && b + k < n) loc[k] = hist[b + k];
        s += loc[k];
    }
    int inc = s;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) wsum[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        int v = wsum[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, v, o);
            if (lane >= o) v += t;
        }
        wsum[lane] = v;
    }
    __syncthreads();
    int run = inc - s + (wid ? wsum[wid - 1] : 0);
#pragma unroll
    for (int k = 0; k < 8; ++k)
        if (k < per && b + k < n) {
            hist[b + k] = run;
            run += loc[k];
        }
}

// scatter walkers to sorted positions; padding positions get perm = -1 and an empty band
__global__ void __launch_bounds__(256)
k_scatter(int n_w, int n_wp, const int *__restrict__ key_w, const int *__restrict__ ilo_w, const int *__restrict__ ihi_w,
          int *__restrict__ offs, int *__restrict__ perm, int *__restrict__ ilo_s, int *__restrict__ ihi_s)
{
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w < n_w) {
        const int pos = atomicAdd(&offs[key_w[w]], 1);
        perm[pos] = w;
        ilo_s[pos] = ilo_w[w];
        ihi_s[pos] = ihi_w[w];
    } else if (w < n_wp) {
        perm[w] = -1;
        ilo_s[w] = 0;
        ihi_s[w] = 0;
    }
}

// ---------------------------------------------------------------------------------------------------
// F1: node amplitude / phase of the stand-in waveform             (Eq. 7; reading R9)
//   A_lm(f)   = c_lm f^(-7/6)/D taper(2f/(m f_ISCO))
//   Psi_lm(f) = (m/2) Psi(2f/m),  Psi(f) = 2 pi f t_c - phi_c - pi/4 + 3/(128 eta (pi M f)^(5/3))
// Phase is written in quarter cycles: y = Psi_lm * 2/pi = 4 f t_c - (m/pi)(phi_c + pi/4) + (m/pi) K (2f/m)^(-5/3).
// Node tables (host-built, per node set): cfp[m][j] = c_lm f_j^(-7/6), f2m[m][j] = 2 f_j/m,
// fm53[m][j] = (2 f_j/m)^(-5/3), f4[j] = 4 f_j.
// ---------------------------------------------------------------------------------------------------
struct NodeTables {
    const double *xj;    // [n]
    const double *hj;    // [n-1]
    const double *invh;  // [n-1]
    const double *ta;    // [n] sub-diagonal of the natural-spline system
    const double *tcp;   // [n] Thomas c'
    const double *tinv;  // [n] Thomas 1/denominator
    const double *f4;    // [n]
    const double *cfp;   // [n_m][n]
    const double *f2m;   // [n_m][n]
    const double *fm53;  // [n_m][n]
    const int *bstart;   // [n]: interval j covers dense bins [bstart[j], bstart[j+1]), j = 0..n-2
    int bc;              // 0 natural, 1 not-a-knot (the tables above are then those of the substituted system)
    double rho0, rhon;   // not-a-knot: M_0 = (1+rho0) M_1 - rho0 M_2,  M_{n-1} = (1+rhon) M_{n-2} - rhon M_{n-3}
};

struct WalkerConst { // per walker constants of the stand-in
    double tc, invD, inv_fisco, K, phi;
};

__device__ __forceinline__ WalkerConst standin_consts(const double *p)
{
    WalkerConst c;
    double Mtot, eta, fi;
    standin_masses(p[0], p[1], Mtot, eta, fi);
    c.tc = p[2];
    c.phi = p[3];
    c.invD = p[4];
    c.inv_fisco = 1.0 / fi;
    const double v = cbrt(kPi * Mtot);
    const double v2 = v * v;
    c.K = 3.0 / (128.0 * eta * (v2 * v2 * v));
    return c;
}

constexpr int kNodesPerThread = 8;

__global__ void __launch_bounds__(128)
k_nodes_standin(const double *__restrict__ params, int P, const int *__restrict__ perm, int n_wp, int n_nodes,
                StandinInfo si, NodeTables nt, double *__restrict__ Y, double *__restrict__ TF)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_wp) return;
    const int j0 = blockIdx.y * kNodesPerThread;
    const int w = perm[p];
    WalkerConst c = {0, 0, 0, 0, 0};
    const double *row = nullptr;
    if (w >= 0) {
        row = params + (size_t)w * P;
        c = standin_consts(row);
    }
    const double inv_kappa = 1.0 / si.kappa;
    for (int m = 0; m < si.n_m; ++m) {
        const double mh_pi = (double)si.mode_m[m] / kPi;
        const double phq = mh_pi * (c.phi + 0.25 * kPi);
        const double Kq = mh_pi * c.K;
        double *ya = Y + ((size_t)(2 * m) * n_nodes) * n_wp + p;
        double *yp = Y + ((size_t)(2 * m + 1) * n_nodes) * n_wp + p;
#pragma unroll
        for (int jj = 0; jj < kNodesPerThread; ++jj) {
            const int j = j0 + jj;
            if (j >= n_nodes) break;
            double a = 0.0, y = 0.0;
            if (w >= 0) {
                const size_t t = (size_t)m * n_nodes + j;
                a = nt.cfp[t] * c.invD * taper(nt.f2m[t] * c.inv_fisco, si.kappa, inv_kappa);
                y = fma(nt.f4[j], c.tc, fma(Kq, nt.fm53[t], -phq));
            }
            ya[(size_t)j * n_wp] = a;
            yp[(size_t)j * n_wp] = y;
        }
        if (blockIdx.y == 0) {
#pragma unroll
            for (int q = 0; q < 4; ++q)
                TF[((size_t)m * 4 + q) * n_wp + p] = (w >= 0) ? row[5 + m * 4 + q] : 0.0;
        }
    }
}

// F1 utility: the stand-in's node arrays in the CALLER layout amp, phase [n_w][n_m][n_nodes] (phase in radians),
// e.g. to feed ll_full_batch / ll_full_batch_tf or ll_tlm_nodes.  One block per walker.
__global__ void __launch_bounds__(128)
k_standin_nodes_out(const double *__restrict__ params, int P, int n_nodes, StandinInfo si, NodeTables nt, GridInfo g,
                    double *__restrict__ amp, double *__restrict__ phase, double *__restrict__ band)
{
    const size_t w = blockIdx.x;
    const WalkerConst c = standin_consts(params + w * P);
    if (band && threadIdx.x == 0) { // the walker's band exactly as k_band_prep takes it (reading R10)
        double Mtot, eta, fi;
        standin_masses(params[w * P], params[w * P + 1], Mtot, eta, fi);
        const double top = (1.0 + si.kappa) * fi * (0.5 * (double)si.m_max);
        const double f_last = bin_freq(g.k_min, g.n_f - 1, g.df);
        band[2 * w] = bin_freq(g.k_min, 0, g.df);
        band[2 * w + 1] = (top < f_last) ? top : f_last;
    }
    const double inv_kappa = 1.0 / si.kappa;
    for (int m = 0; m < si.n_m; ++m) {
        const double mh_pi = (double)si.mode_m[m] / kPi;
        const double phq = mh_pi * (c.phi + 0.25 * kPi);
        const double Kq = mh_pi * c.K;
        for (int j = threadIdx.x; j < n_nodes; j += blockDim.x) {
            const size_t t = (size_t)m * n_nodes + j;
            const size_t o = (w * si.n_m + m) * n_nodes + j;
            amp[o] = nt.cfp[t] * c.invD * taper(nt.f2m[t] * c.inv_fisco, si.kappa, inv_kappa);
            phase[o] = fma(nt.f4[j], c.tc, fma(Kq, nt.fm53[t], -phq)) * kPio2_1; // quarter cycles -> radians
        }
    }
}

// F1 (array entry point): transpose caller arrays [n_w][n_m][n_nodes] into Y; phase radians -> quarter cycles
__global__ void __launch_bounds__(256)
k_nodes_arrays(const double *__restrict__ amp, const double *__restrict__ phase, const double *__restrict__ tf,
               const int *__restrict__ perm, int n_wp, int n_nodes, int n_m, double *__restrict__ Y,
               double *__restrict__ TF)
{
    __shared__ double ta[32][33], tp[32][33];
    const int m = blockIdx.z;
    const int p0 = blockIdx.x * 32, j0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5; // 32 x 8
    for (int r = ty; r < 32; r += 8) {
        const int w = perm[p0 + r];
        const int j = j0 + tx;
        double a = 0.0, ph = 0.0;
        if (w >= 0 && j < n_nodes) {
            const size_t idx = ((size_t)w * n_m + m) * n_nodes + j;
            a = amp[idx];
            ph = phase[idx] * kTwoOverPi;
        }
        ta[r][tx] = a;
        tp[r][tx] = ph;
    }
    __syncthreads();
    for (int r = ty; r < 32; r += 8) {
        const int j = j0 + r;
        if (j < n_nodes) {
            Y[((size_t)(2 * m) * n_nodes + j) * n_wp + p0 + tx] = ta[tx][r];
            Y[((size_t)(2 * m + 1) * n_nodes + j) * n_wp + p0 + tx] = tp[tx][r];
        }
    }
    if (blockIdx.y == 0 && threadIdx.x < 32) {
        const int w = perm[p0 + tx];
#pragma unroll
        for (int q = 0; q < 4; ++q)
            TF[((size_t)m * 4 + q) * n_wp + p0 + tx] = (w >= 0) ? tf[((size_t)w * n_m + m) * 4 + q] : 0.0;
    }
}

// F1 (array entry point with a frequency-dependent transfer function, Eq. 8-9): six splines per mode,
// sys = 6 m + s with s = 0 amplitude, 1 phase (radians -> quarter cycles), 2 + 2c Re T^c, 3 + 2c Im T^c;
// tf_nodes is [n_w][n_m][n_c][n_nodes][2].  One 32 x 32 transpose tile per block, blockIdx.z = sys.
__global__ void __launch_bounds__(256)
k_nodes_arrays_tf(const double *__restrict__ amp, const double *__restrict__ phase, const double *__restrict__ tf_nodes,
                  const int *__restrict__ perm, int n_wp, int n_nodes, int n_m, double *__restrict__ Y)
{
    __shared__ double tt[32][33];
    const int sys = blockIdx.z, m = sys / 6, s = sys % 6;
    const int p0 = blockIdx.x * 32, j0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5; // 32 x 8
    for (int r = ty; r < 32; r += 8) {
        const int w = perm[p0 + r];
        const int j = j0 + tx;
        double v = 0.0;
        if (w >= 0 && j < n_nodes) {
            const size_t wm = (size_t)w * n_m + m;
            if (s == 0) v = amp[wm * n_nodes + j];
            else if (s == 1) v = phase[wm * n_nodes + j] * kTwoOverPi;
            else v = tf_nodes[((wm * kNC + ((s - 2) >> 1)) * n_nodes + j) * 2 + ((s - 2) & 1)];
        }
        tt[r][tx] = v;
    }
    __syncthreads();
    for (int r = ty; r < 32; r += 8) {
        const int j = j0 + r;
        if (j < n_nodes) Y[((size_t)sys * n_nodes + j) * n_wp + p0 + tx] = tt[tx][r];
    }
}

// ---------------------------------------------------------------------------------------------------
// F2: natural cubic spline, one system per thread, systems interleaved so every load/store is coalesced.
// The tridiagonal matrix depends only on the (shared) nodes, so its Thomas factorisation (ta, tcp, tinv) is
// built once per node set on the host; per system only the two substitution sweeps remain   (reading R1):
//   dp_j = (r_j - a_j dp_{j-1}) / den_j,   r_j = (y_{j+1}-y_j)/h_j - (y_j-y_{j-1})/h_{j-1}
//   M_j  = dp_j - c'_j M_{j+1},            M_0 = M_{n-1} = 0
//   b_j = (y_{j+1}-y_j)/h_j - h_j (2 M_j + M_{j+1})/6,  c_j = M_j/2,  d_j = (M_{j+1}-M_j)/(6 h_j)
// dp_j is parked in the b-slot of interval j between the sweeps.
// ---------------------------------------------------------------------------------------------------
constexpr int kSplineBlk = 16;
__global__ void __launch_bounds__(128)
k_spline(const double *__restrict__ Y, double *__restrict__ C, int n_wp, int n_nodes, int n_m, int ns, NodeTables nt)
{
    // ns = splines per mode: 2 (amplitude, phase) or 6 (+ Re/Im of T^A, T^E: frequency-dependent transfer function)
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_wp) return;
    const int sys = blockIdx.y, m = sys / ns, kind = sys % ns;
    const size_t sw = (size_t)n_wp;
    const double *y = Y + (size_t)sys * n_nodes * sw + p;
    double *c = C + ((size_t)m * ns * 4 + kind * 4) * sw + p; // + j * (n_m*ns*4*sw) + q*sw
    const size_t cj = (size_t)n_m * ns * 4 * sw;
    const int n = n_nodes;

    double yprev = __ldg(y), ycur = __ldg(y + sw);
    double sprev = (ycur - yprev) * __ldg(nt.invh);
    double dpp = 0.0;
    // node values are read through the read-only path (__ldg): the compiler may then hoist the loads of an
    // unrolled group above the stores of the parked dp values instead of paying one memory latency per row
#pragma unroll 16
    for (int j = 1; j <= n - 2; ++j) {
        const double ynext = __ldg(y + (size_t)(j + 1) * sw);
        const double s = (ynext - ycur) * __ldg(nt.invh + j);
        const double r = s - sprev;
        const double dp = (r - __ldg(nt.ta + j) * dpp) * __ldg(nt.tinv + j);
        c[(size_t)j * cj + sw] = dp;
        dpp = dp;
        sprev = s;
        ycur = ynext;
    }
    // backward sweep in register blocks of kSplineBlk intervals: the parked dp values and node values of a
    // block are loaded first (independent loads, all in flight together), then the recurrence runs on
    // registers, then the coefficients are stored.  (A load of dp_j issued between the stores of interval
    // j + 1 could not be hoisted by the compiler: same base pointer, so each step paid a full memory latency.)
    double Mn = 0.0, Mnn = 0.0; // M_{j+1}, M_{j+2}
    if (nt.bc) { // not-a-knot: M_{n-1} from M_{n-2} = dp_{n-2} (its c' is 0) and M_{n-3}
        const double M2 = c[(size_t)(n - 2) * cj + sw];
        const double M3 = fma(-__ldg(nt.tcp + n - 3), M2, c[(size_t)(n - 3) * cj + sw]);
        Mn = (1.0 + nt.rhon) * M2 - nt.rhon * M3;
    }
    double y1 = __ldg(y + (size_t)(n - 1) * sw);
    for (int jt = n - 2; jt >= 0; jt -= kSplineBlk) {
        double dpv[kSplineBlk], yv[kSplineBlk];
#pragma unroll
        for (int k = 0; k < kSplineBlk; ++k) {
            const int j = jt - k;
            dpv[k] = (j >= 1) ? c[(size_t)j * cj + sw] : 0.0;
            yv[k] = (j >= 0) ? __ldg(y + (size_t)j * sw) : 0.0;
        }
#pragma unroll
        for (int k = 0; k < kSplineBlk; ++k) {
            const int j = jt - k;
            if (j >= 0) {
                const double y0 = yv[k];
                const double Mj = (j >= 1) ? fma(-__ldg(nt.tcp + j), Mn, dpv[k])
                                           : (nt.bc ? (1.0 + nt.rho0) * Mn - nt.rho0 * Mnn : 0.0);
                const double h = __ldg(nt.hj + j), ih = __ldg(nt.invh + j);
                double *cc = c + (size_t)j * cj;
                cc[0] = y0;
                cc[sw] = (y1 - y0) * ih - h * (2.0 * Mj + Mn) * kSixth;
                cc[2 * sw] = 0.5 * Mj;
                cc[3 * sw] = (Mn - Mj) * ih * kSixth;
                Mnn = Mn;
                Mn = Mj;
                y1 = y0;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// F2 for small batches (Module-1 sized: tens to hundreds of walkers): one warp or block per system.  With
// few systems the thread-per-system kernel above is a chain of 2 (n-2) dependent steps on a nearly empty GPU.
// Both Thomas sweeps are first-order linear recurrences x_j = alpha_j + beta_j x_{j-1}, i.e. compositions of
// affine maps, which are associative: each thread composes the maps of its ceil(n/T) consecutive rows, a scan
// composes across threads, and each thread then re-runs its rows from the right start value.  Dependent chain:
// 2 ceil(n/T) + scan steps instead of n.  Same factorisation tables; results differ from the sequential sweep
// by rounding only.  Shared memory per warp: node values and dp / M, 2 n doubles.
// ---------------------------------------------------------------------------------------------------
// Generalised to one BLOCK of T = 32..256 threads per system (T ~ n/4): the scan runs inside each warp and then
// across the warps' totals, so 1024 nodes are a chain of 2 x 4 rows + two block scans instead of 2 x 32 rows.
__device__ __forceinline__ void affine_block_scan_up(double &A, double &B, double *sA, double *sB, int lane, int wid, int nwarp)
{
    // inclusive scan of maps x -> A + B x in thread order (thread t's map applied after those of threads < t)
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const double Ap = __shfl_up_sync(0xffffffffu, A, o), Bp = __shfl_up_sync(0xffffffffu, B, o);
        if (lane >= o) { A = fma(B, Ap, A); B *= Bp; }
    }
    if (nwarp > 1) {
        if (lane == 31) { sA[wid] = A; sB[wid] = B; }
        __syncthreads();
        double pa = 0.0, pb = 1.0; // composition of the warps below, in order
        for (int k = 0; k < wid; ++k) { pa = fma(sB[k], pa, sA[k]); pb *= sB[k]; }
        A = fma(B, pa, A);
        B *= pb;
        __syncthreads();
    }
}
__device__ __forceinline__ void affine_block_scan_down(double &A, double &B, double *sA, double *sB, int lane, int wid, int nwarp)
{
    // the mirror image: thread t's map applied after those of threads > t
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const double Ap = __shfl_down_sync(0xffffffffu, A, o), Bp = __shfl_down_sync(0xffffffffu, B, o);
        if (lane + o < 32) { A = fma(B, Ap, A); B *= Bp; }
    }
    if (nwarp > 1) {
        if (lane == 0) { sA[wid] = A; sB[wid] = B; }
        __syncthreads();
        double pa = 0.0, pb = 1.0;
        for (int k = nwarp - 1; k > wid; --k) { pa = fma(sB[k], pa, sA[k]); pb *= sB[k]; }
        A = fma(B, pa, A);
        B *= pb;
        __syncthreads();
    }
}

__global__ void __launch_bounds__(256)
k_spline_block(const double *__restrict__ Y, double *__restrict__ C, int n_wp, int n_nodes, int n_m, int ns, NodeTables nt)
{
    extern __shared__ double ssm[]; // ys[n], ds[n], then the exchange slots
    __shared__ double sA[8], sB[8];
    const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31, wid = tid >> 5, nwarp = T >> 5;
    const int sys = blockIdx.x / n_wp, p = blockIdx.x - sys * n_wp;
    const int m = sys / ns, kind = sys % ns;
    const int n = n_nodes;
    const size_t sw = (size_t)n_wp;
    double *ys = ssm, *ds = ys + n, *xch = ds + n; // xch[T]: value handed to the neighbouring thread
    for (int j = tid; j < n; j += T) ys[j] = __ldg(Y + ((size_t)sys * n + j) * sw + p);
    __syncthreads();
    const int L = (n + T - 1) / T;
    const int j0 = min(tid * L, n), j1 = min(j0 + L, n);
    auto rhs = [&](int j) { return (ys[j + 1] - ys[j]) * __ldg(nt.invh + j) - (ys[j] - ys[j - 1]) * __ldg(nt.invh + j - 1); };
    // ---- forward sweep: dp_j = (r_j - a_j dp_{j-1}) / den_j for j = 1..n-2, dp_0 = 0
    double A = 0.0, B = 1.0;
    for (int j = j0; j < j1; ++j)
        if (j >= 1 && j <= n - 2) {
            const double ti = __ldg(nt.tinv + j), be = -__ldg(nt.ta + j) * ti;
            A = fma(be, A, rhs(j) * ti);
            B *= be;
        }
    affine_block_scan_up(A, B, sA, sB, lane, wid, nwarp);
    xch[tid] = A; // all maps up to and including this thread applied to dp_0 = 0
    __syncthreads();
    double start = tid ? xch[tid - 1] : 0.0;
    for (int j = j0; j < j1; ++j) {
        if (j >= 1 && j <= n - 2) start = (rhs(j) - __ldg(nt.ta + j) * start) * __ldg(nt.tinv + j);
        ds[j] = (j >= 1 && j <= n - 2) ? start : 0.0;
    }
    __syncthreads();
    // ---- backward sweep: M_j = dp_j - c'_j M_{j+1} for j = n-2..1, M_0 = M_{n-1} = 0
    A = 0.0; B = 1.0;
    for (int j = j1 - 1; j >= j0; --j) {
        if (j >= 1 && j <= n - 2) {
            const double be = -__ldg(nt.tcp + j);
            A = fma(be, A, ds[j]);
            B *= be;
        } else { A = 0.0; B = 0.0; }
    }
    affine_block_scan_down(A, B, sA, sB, lane, wid, nwarp);
    xch[tid] = A;
    __syncthreads();
    double Mn = (tid + 1 < T) ? xch[tid + 1] : 0.0;
    for (int j = j1 - 1; j >= j0; --j) {
        Mn = (j >= 1 && j <= n - 2) ? fma(-__ldg(nt.tcp + j), Mn, ds[j]) : 0.0;
        ds[j] = Mn;
    }
    __syncthreads();
    if (nt.bc) { // not-a-knot end values from their neighbours
        if (tid == 0) {
            ds[0] = (1.0 + nt.rho0) * ds[1] - nt.rho0 * ds[2];
            ds[n - 1] = (1.0 + nt.rhon) * ds[n - 2] - nt.rhon * ds[n - 3];
        }
        __syncthreads();
    }
    // ---- coefficients of interval j (same formulas as k_spline)
    double *c = C + ((size_t)m * ns * 4 + kind * 4) * sw + p;
    const size_t cj = (size_t)n_m * ns * 4 * sw;
    for (int j = tid; j < n - 1; j += T) {
        const double y0 = ys[j], y1 = ys[j + 1], Mj = ds[j], Mn1 = ds[j + 1];
        const double h = __ldg(nt.hj + j), ih = __ldg(nt.invh + j);
        double *cc = c + (size_t)j * cj;
        cc[0] = y0;
        cc[sw] = (y1 - y0) * ih - h * (2.0 * Mj + Mn1) * kSixth;
        cc[2 * sw] = 0.5 * Mj;
        cc[3 * sw] = (Mn1 - Mj) * ih * kSixth;
    }
}

// ---------------------------------------------------------------------------------------------------
// F3: fused spline evaluation / channel response / inner products           (Eq. 3, 7, 9)
// One thread = one walker; a warp = 32 walkers walking the SAME dense bins, so the data tile (g4, W) is a
// shared-memory broadcast and no cross-thread reduction exists.  Tiles of g4/W arrive by 1-D bulk TMA into
// a two-stage ring guarded by mbarriers.  The dense template is never written anywhere.
// Single-mode specialisation: T^c is constant per walker, so the kernel accumulates the complex sums
// S^c = sum_i g^c_i A e^{-i Psi} and H = sum_i W_i A^2; k_finalize applies T^c.
// ---------------------------------------------------------------------------------------------------
struct FusedArgs {
    const double *g4;
    const double *Wd;
    const double *C;
    const double *TF;
    const double *xj;
    const int *bstart;
    const int *ilo;
    const int *ihi;
    double *part;
    long long k_min;
    double df;
    const int *tile_start; // [n_tiles + 1]: frequency tile t covers dense bins [tile_start[t], tile_start[t+1])
    int n_f, n_wp, n_nodes, n_m, TB, CH;
};

// largest t in [0, n_tiles-1] with tile_start[t] <= i
__device__ __forceinline__ int tile_of_bin(const int *__restrict__ tile_start, int n_tiles, int i)
{
    int lo = 0, hi = n_tiles - 1;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (__ldg(tile_start + mid) <= i) lo = mid; else hi = mid - 1;
    }
    return lo;
}

__device__ __forceinline__ int find_interval_of_bin(const int *__restrict__ bstart, int n_nodes, int i)
{
    // largest j in [0, n-2] with bstart[j] <= i
    int lo = 0, hi = n_nodes - 2;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (__ldg(bstart + mid) <= i) lo = mid; else hi = mid - 1;
    }
    return lo;
}

#ifndef LL_FUSED_UNROLL
#define LL_FUSED_UNROLL 3 // bins in flight per thread in the hot loop (tuned on B200, profiles/)
#endif
#ifndef LL_FUSED_MINB
#define LL_FUSED_MINB 4 // resident 128-thread blocks per SM the register budget is held to
#endif
constexpr int kFusedUnroll = LL_FUSED_UNROLL;
// bins [b0, b1) of one spline interval for the single-mode kernel: t, the two cubics, A e^{-i Psi}, the two
// complex MACs with g^A, g^E and W A^2.  MASK = per-lane band test (only at the ragged ends of a warp's band).
template <bool MASK>
__device__ __forceinline__ void fused_bins_nm1(int b0, int b1, int tlo, int thi, int kbase, double df, double nxj,
                                               double cA0, double cA1, double cA2, double cA3, double cP0, double cP1,
                                               double cP2, double cP3, const double4 *__restrict__ sg4,
                                               const double *__restrict__ sWc, double &sAr, double &sAi, double &sEr,
                                               double &sEi, double &sH)
{
#pragma unroll kFusedUnroll
    for (int ii = b0; ii < b1; ++ii) {
        const double t = fma((double)(kbase + ii), df, nxj);
        double A = fma(fma(fma(cA3, t, cA2), t, cA1), t, cA0);
        const double y = fma(fma(fma(cP3, t, cP2), t, cP1), t, cP0);
        if (MASK) A = ((ii >= tlo) && (ii < thi)) ? A : 0.0;
        double u, v; // h = u - i v
        amp_expi_qc(A, y, u, v);
        const double4 g = sg4[ii];
        const double w = sWc[ii];
        sAr = fma(g.x, u, sAr); sAr = fma(g.y, v, sAr);
        sAi = fma(g.y, u, sAi); sAi = fma(-g.x, v, sAi);
        sEr = fma(g.z, u, sEr); sEr = fma(g.w, v, sEr);
        sEi = fma(g.w, u, sEi); sEi = fma(-g.z, v, sEi);
        sH = fma(w * A, A, sH);
    }
}

// The same bins by recurrence (SURVEY.md "hard parts"; unmasked bins of one spline interval only).  On the uniform
// grid the phase cubic has constant third differences, so e^{-i Psi_k} advances by three complex rotations per bin,
//   z_{k+1} = z_k w_k,  w_{k+1} = w_k v_k,  v_{k+1} = v_k u,   w = e^{i D1 Psi}, v = e^{i D2 Psi}, u = e^{i D3 Psi},
// and the amplitude cubic by its forward differences; every kRotSync bins everything is re-evaluated from the cubic
// coefficients (the exact route above), which bounds the accumulated rounding: with D1 Psi <= a few quarter cycles
// known to 1 ulp, the phase drifts by < kRotSync^2/2 ulp ~ 1e-13 quarter cycles between re-syncs, far below the
// rounding of Psi itself (1e-9 at 1e7 quarter cycles).  Per bin: 12 (rotations) + 3 (amplitude) + 2 (A z) + 8
// (MACs) + 2 (W A^2) = 27 FP64 instructions and no sincos, no quadrant fix-up, no bin-number conversion, instead of
// 34 + 18 others.
#ifndef LL_FUSED_ROT
#define LL_FUSED_ROT 1
#endif
#ifndef LL_ROT_SYNC
#define LL_ROT_SYNC 32 // measured at config 2 (max |error of <d|h>| over sampled walkers, kernel time): 32: 8e-8, 10.7 ms
                       // (the exact route: 7e-8, 13.0 ms); 64: 3e-7, 10.2 ms; 128: 2e-6, 10.0 ms; 256: 1.3e-5, 9.9 ms
#endif
#ifndef LL_ROT_UNROLL
#define LL_ROT_UNROLL 2
#endif
constexpr int kRotSync = LL_ROT_SYNC;
constexpr int kRotUnroll = LL_ROT_UNROLL;
// The sin/cos polynomials are minimax fits: cos(0) comes out as 1 - 5.5e-14, so a rotation built from them has modulus
// 1 - O(1e-14).  Harmless once, but u multiplies into v, v into w and w into z every bin, and the modulus of z would
// decay like k^3/6 x 5.5e-14 (measured: 5e-10 relative on <d|h> at 64 bins between re-syncs).  One Newton step of
// 1/sqrt(c^2 + s^2) around 1 restores the unit modulus to rounding.
__device__ __forceinline__ void unit_modulus(double &c, double &s)
{
    const double k = fma(-0.5, fma(c, c, s * s), 1.5);
    c *= k;
    s *= k;
}
__device__ __forceinline__ void fused_bins_rot(int b0, int b1, int kbase, double df, double nxj, double cA0, double cA1,
                                               double cA2, double cA3, double cP0, double cP1, double cP2, double cP3,
                                               const double4 *__restrict__ sg4, const double *__restrict__ sWc,
                                               double &sAr, double &sAi, double &sEr, double &sEi, double &sH)
{
    const double df2 = df * df, df3 = df2 * df;
    const double d3A = 6.0 * cA3 * df3;
    double su, cu;
    sincos_qc(6.0 * cP3 * df3, su, cu);
    unit_modulus(cu, su);
    for (int k0 = b0; k0 < b1; k0 += kRotSync) {
        const int k1 = min(k0 + kRotSync, b1);
        const double t = fma((double)(kbase + k0), df, nxj);
        // f(t), f(t+df) - f(t) = df [c1 + c2 (2t + df) + c3 (3t^2 + 3t df + df^2)], second difference df^2 [2 c2 + 6 c3 (t + df)]
        const double tt = fma(2.0, t, df), q3 = fma(3.0 * t, t + df, df2), t1 = t + df;
        double A = fma(fma(fma(cA3, t, cA2), t, cA1), t, cA0);
        double d1A = df * fma(cA3, q3, fma(cA2, tt, cA1));
        double d2A = df2 * fma(6.0 * cA3, t1, 2.0 * cA2);
        double sz, cz, sw, cw, sv, cv;
        sincos_qc(fma(fma(fma(cP3, t, cP2), t, cP1), t, cP0), sz, cz);
        sincos_qc(df * fma(cP3, q3, fma(cP2, tt, cP1)), sw, cw);
        sincos_qc(df2 * fma(6.0 * cP3, t1, 2.0 * cP2), sv, cv);
        unit_modulus(cz, sz);
        unit_modulus(cw, sw);
        unit_modulus(cv, sv);
#pragma unroll kRotUnroll
        for (int ii = k0; ii < k1; ++ii) {
            const double u = A * cz, v = A * sz; // h = u - i v
            const double4 g = sg4[ii];
            const double w = sWc[ii];
            sAr = fma(g.x, u, sAr); sAr = fma(g.y, v, sAr);
            sAi = fma(g.y, u, sAi); sAi = fma(-g.x, v, sAi);
            sEr = fma(g.z, u, sEr); sEr = fma(g.w, v, sEr);
            sEi = fma(g.w, u, sEi); sEi = fma(-g.z, v, sEi);
            sH = fma(w * A, A, sH);
            const double nzc = fma(cz, cw, -(sz * sw)), nzs = fma(sz, cw, cz * sw);
            const double nwc = fma(cw, cv, -(sw * sv)), nws = fma(sw, cv, cw * sv);
            const double nvc = fma(cv, cu, -(sv * su)), nvs = fma(sv, cu, cv * su);
            cz = nzc; sz = nzs; cw = nwc; sw = nws; cv = nvc; sv = nvs;
            A += d1A; d1A += d2A; d2A += d3A;
        }
    }
}

template <int NM1> // NM1 = 1: single-mode specialisation (NQ = 5); 0: any n_m (NQ = 2)
__global__ void __launch_bounds__(128, LL_FUSED_MINB) k_full_fused(FusedArgs a)
{
    extern __shared__ __align__(128) double sm[];
    __shared__ __align__(8) uint64_t bar[2];
    __shared__ int s_lo, s_hi;

    const int tid = threadIdx.x;
    const int p = blockIdx.x * blockDim.x + tid;
    const int tile = blockIdx.y;
    const int i0 = __ldg(a.tile_start + tile), i1 = __ldg(a.tile_start + tile + 1); // tile = dense bins [i0, i1)
    const int lo = max(a.ilo[p], i0), hi = min(a.ihi[p], i1);
    if (tid == 0) {
        s_lo = INT_MAX;
        s_hi = INT_MIN;
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (lo < hi) {
        atomicMin(&s_lo, lo);
        atomicMax(&s_hi, hi);
    }
    __syncthreads();
    const int blo = s_lo, bhi = s_hi;
    if (blo >= bhi) return; // no walker of this block has bins in this tile; k_finalize never reads it

    const int CH = a.CH;
    const int c_begin = blo / CH, c_end = (bhi + CH - 1) / CH;
    const uint32_t stage_bytes = (uint32_t)CH * 40u;
    auto issue = [&](int c, int st) {
        double *dst = sm + (size_t)st * CH * 5;
        mbar_expect_tx(&bar[st], stage_bytes);
        tma_load_1d(dst, a.g4 + (size_t)c * CH * 4, (uint32_t)CH * 32u, &bar[st]);
        tma_load_1d(dst + (size_t)CH * 4, a.Wd + (size_t)c * CH, (uint32_t)CH * 8u, &bar[st]);
    };
    if (tid == 0) issue(c_begin, 0);

    const size_t sw = (size_t)a.n_wp;
    const size_t cj = (size_t)a.n_m * 8 * sw;
    int j = find_interval_of_bin(a.bstart, a.n_nodes, blo);
    int jl = -1;
    double cA0 = 0, cA1 = 0, cA2 = 0, cA3 = 0, cP0 = 0, cP1 = 0, cP2 = 0, cP3 = 0, nxj = 0;
    const int kbase = (int)a.k_min; // k_min + n_f < 2^31 is checked on the host
    double sAr = 0, sAi = 0, sEr = 0, sEi = 0, sH = 0; // NM1: S^A, S^E, H;  generic: sAr = d_h, sH = h_h

    for (int c = c_begin; c < c_end; ++c) {
        const int st = (c - c_begin) & 1;
        const uint32_t ph = (uint32_t)((c - c_begin) >> 1) & 1u;
        if (tid == 0 && c + 1 < c_end) issue(c + 1, st ^ 1);
        mbar_wait(&bar[st], ph);
        const double *sg = sm + (size_t)st * CH * 5;
        const double *sW = sg + (size_t)CH * 4;
        const int cb = c * CH;
        const int ce = min(cb + CH, bhi);
        int i = max(cb, blo);
        while (i < ce) {
            while (j < a.n_nodes - 2 && __ldg(a.bstart + j + 1) <= i) ++j;
            const int seg_end = (j < a.n_nodes - 2) ? min(__ldg(a.bstart + j + 1), ce) : ce;
            int tlo = max(i, lo), thi = min(seg_end, hi);
            if (tlo >= thi) { tlo = INT_MAX; thi = INT_MIN; }
            const int wlo = __reduce_min_sync(0xffffffffu, tlo);
            const int whi = __reduce_max_sync(0xffffffffu, thi);
            if (wlo < whi) {
                if (NM1) {
                    if (j != jl) {
                        const double *cc = a.C + (size_t)j * cj + p;
                        cA0 = cc[0]; cA1 = cc[sw]; cA2 = cc[2 * sw]; cA3 = cc[3 * sw];
                        cP0 = cc[4 * sw]; cP1 = cc[5 * sw]; cP2 = cc[6 * sw]; cP3 = cc[7 * sw];
                        nxj = -__ldg(a.xj + j);
                        jl = j;
                    }
                    // bins every lane of the warp has inside its band run without the per-lane mask
                    const int flo = __reduce_max_sync(0xffffffffu, max(lo, i));
                    const int fhi = __reduce_min_sync(0xffffffffu, min(hi, seg_end));
                    const double4 *sg4 = reinterpret_cast<const double4 *>(sg) - cb;
                    const double *sWc = sW - cb;
                    if (flo < fhi) {
                        fused_bins_nm1<true>(wlo, flo, tlo, thi, kbase, a.df, nxj, cA0, cA1, cA2, cA3, cP0, cP1, cP2, cP3,
                                             sg4, sWc, sAr, sAi, sEr, sEi, sH);
                        if (LL_FUSED_ROT && fhi - flo >= 8)
                            fused_bins_rot(flo, fhi, kbase, a.df, nxj, cA0, cA1, cA2, cA3, cP0, cP1, cP2, cP3, sg4, sWc,
                                           sAr, sAi, sEr, sEi, sH);
                        else
                            fused_bins_nm1<false>(flo, fhi, tlo, thi, kbase, a.df, nxj, cA0, cA1, cA2, cA3, cP0, cP1, cP2, cP3,
                                                  sg4, sWc, sAr, sAi, sEr, sEi, sH);
                        fused_bins_nm1<true>(fhi, whi, tlo, thi, kbase, a.df, nxj, cA0, cA1, cA2, cA3, cP0, cP1, cP2, cP3,
                                             sg4, sWc, sAr, sAi, sEr, sEi, sH);
                    } else {
                        fused_bins_nm1<true>(wlo, whi, tlo, thi, kbase, a.df, nxj, cA0, cA1, cA2, cA3, cP0, cP1, cP2, cP3,
                                             sg4, sWc, sAr, sAi, sEr, sEi, sH);
                    }
                } else {
                    // any number of modes: chunks of four bins with the MODE loop outside the bins, so that a mode's
                    // 8 coefficients and 4 transfer factors are read once per chunk (not once per bin) and the four
                    // bins are four independent cubic -> sincos -> T^c h chains in flight per thread
                    nxj = -__ldg(a.xj + j);
                    const double *cc0 = a.C + (size_t)j * cj + p;
                    for (int c4 = wlo; c4 < whi; c4 += 4) {
                        double t4[4], h4[4][4];
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            t4[k] = fma((double)(kbase + c4 + k), a.df, nxj);
                            h4[k][0] = h4[k][1] = h4[k][2] = h4[k][3] = 0.0;
                        }
#pragma unroll 1
                        for (int m = 0; m < a.n_m; ++m) {
                            const double *cc = cc0 + (size_t)m * 8 * sw;
                            double co[8];
#pragma unroll
                            for (int q = 0; q < 8; ++q) co[q] = cc[(size_t)q * sw];
                            const double *tf = a.TF + (size_t)m * 4 * sw + p;
                            const double tar = tf[0], tai = tf[sw], ter = tf[2 * sw], tei = tf[3 * sw];
#pragma unroll
                            for (int k = 0; k < 4; ++k) {
                                const double A = fma(fma(fma(co[3], t4[k], co[2]), t4[k], co[1]), t4[k], co[0]);
                                const double y = fma(fma(fma(co[7], t4[k], co[6]), t4[k], co[5]), t4[k], co[4]);
                                double u, v; // h_m = u - i v
                                amp_expi_qc(A, y, u, v);
                                h4[k][0] = fma(tar, u, h4[k][0]); h4[k][0] = fma(tai, v, h4[k][0]);
                                h4[k][1] = fma(tai, u, h4[k][1]); h4[k][1] = fma(-tar, v, h4[k][1]);
                                h4[k][2] = fma(ter, u, h4[k][2]); h4[k][2] = fma(tei, v, h4[k][2]);
                                h4[k][3] = fma(tei, u, h4[k][3]); h4[k][3] = fma(-ter, v, h4[k][3]);
                            }
                        }
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            const int ii = c4 + k;
                            if (ii < whi && ii >= tlo && ii < thi) {
                                const double4 g = reinterpret_cast<const double4 *>(sg)[ii - cb];
                                const double w = sW[ii - cb];
                                sAr = fma(g.x, h4[k][0], sAr); sAr = fma(-g.y, h4[k][1], sAr);
                                sAr = fma(g.z, h4[k][2], sAr); sAr = fma(-g.w, h4[k][3], sAr);
                                sH = fma(w, h4[k][0] * h4[k][0] + h4[k][1] * h4[k][1] + h4[k][2] * h4[k][2] + h4[k][3] * h4[k][3], sH);
                            }
                        }
                    }
                }
            }
            i = seg_end;
        }
        __syncthreads(); // everyone is done with stage st before it is refilled two chunks later
    }
    if (NM1) {
        double *o = a.part + ((size_t)tile * 5) * sw + p;
        o[0] = sAr; o[sw] = sAi; o[2 * sw] = sEr; o[3 * sw] = sEi; o[4 * sw] = sH;
    } else {
        double *o = a.part + ((size_t)tile * 2) * sw + p;
        o[0] = sAr; o[sw] = sH;
    }
}

// ---------------------------------------------------------------------------------------------------
// F3, FP32-accumulate variant (BASELINE.json config 2; reading R15), single mode.
// FP64: bin frequency offset t, phase and amplitude cubics, reduction of the phase to [-1/2, 1/2] quarter
// cycles and its scaling to radians, <h|h> = sum W A^2 (all terms positive: binary32 partial sums would lose
// ~1e-7 of it), every sum longer than kMixedChain terms.  binary32: sin/cos polynomials, A e^{-i Psi}, the
// products with the pre-scaled binary32 data tile and <d|h> partial sums of <= kMixedChain terms.
// The data are pre-scaled by a power of two sigma (g/sigma in binary32, W/sigma^2 in FP64; amplitudes * sigma)
// so that every binary32 quantity is O(1): k_prescale_f32.
// ---------------------------------------------------------------------------------------------------
constexpr int kMixedChain = 8;

// scale[0] = sigma = 2^ceil(log2(max W)/2), scale[1] = 1/sigma, scale[2] = 1/sigma^2 (exact powers of two)
__global__ void __launch_bounds__(256) k_wmax(const double *__restrict__ W, long long n_f, unsigned long long *__restrict__ wmax_bits)
{
    double m = 0.0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_f; i += (long long)gridDim.x * blockDim.x) {
        const double w = fabs(W[i]);
        if (w > m && w < INFINITY) m = w;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) atomicMax(wmax_bits, (unsigned long long)__double_as_longlong(m)); // m >= 0: order-preserving
}
__global__ void k_scale_from_wmax(const unsigned long long *__restrict__ wmax_bits, double *__restrict__ scale)
{
    const double m = __longlong_as_double((long long)wmax_bits[0]);
    int e = 0;
    if (m > 0.0) {
        (void)frexp(m, &e); // m = f 2^e, f in [1/2, 1)
        e = (e + 1) >> 1;   // sigma^2 = 2^(2e) >= m
    }
    scale[0] = ldexp(1.0, e);
    scale[1] = ldexp(1.0, -e);
    scale[2] = ldexp(1.0, -2 * e);
}
__global__ void __launch_bounds__(256) k_prescale_f32(const double *__restrict__ g4, const double *__restrict__ Wd,
                                                      long long n_pad, const double *__restrict__ scale,
                                                      float *__restrict__ g4f, double *__restrict__ Wds)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_pad) return;
    const double is = scale[1], is2 = scale[2];
    const double4 g = reinterpret_cast<const double4 *>(g4)[i];
    // pair-interleaved: bins (2p, 2p+1) -> [Ar Ar' Ai Ai' Er Er' Ei Ei'], so that one LDS.128 pair feeds f32x2 MACs
    float *o = g4f + (i >> 1) * 8 + (i & 1);
    o[0] = (float)(g.x * is); o[2] = (float)(g.y * is); o[4] = (float)(g.z * is); o[6] = (float)(g.w * is);
    Wds[i] = Wd[i] * is2;
}

struct MixedAcc { // FP64 accumulators of one walker
    double sAr, sAi, sEr, sEi, sH;
};

// bins [b0, b1) of one spline interval, in chains of <= kMixedChain bins flushed into the FP64 accumulators
template <bool MASK>
__device__ __forceinline__ void fused_bins_mixed(int b0, int b1, int tlo, int thi, int kbase, double df, double nxj,
                                                 double cA0, double cA1, double cA2, double cA3, double cP0, double cP1,
                                                 double cP2, double cP3, const float *__restrict__ sgp,
                                                 const double *__restrict__ sWc, MixedAcc &acc)
{
    // sgp: pair-interleaved data tile addressed by global bin (see k_prescale_f32)
    for (int base = b0; base < b1; base += kMixedChain) {
        const int end = min(base + kMixedChain, b1);
        float fAr = 0.f, fAi = 0.f, fEr = 0.f, fEi = 0.f;
#pragma unroll 4
        for (int ii = base; ii < end; ++ii) {
            const double t = fma((double)(kbase + ii), df, nxj);
            double A = fma(fma(fma(cA3, t, cA2), t, cA1), t, cA0);
            const double y = fma(fma(fma(cP3, t, cP2), t, cP1), t, cP0);
            if (MASK) A = ((ii >= tlo) && (ii < thi)) ? A : 0.0;
            acc.sH = fma(sWc[ii] * A, A, acc.sH);
            float u, v; // h = u - i v
            amp_expi_qc_f32(__double2float_rn(A), y, u, v);
            const float *gp = sgp + (ii >> 1) * 8 + (ii & 1);
            const float gx = gp[0], gy = gp[2], gz = gp[4], gw = gp[6];
            fAr = fmaf(gx, u, fAr); fAr = fmaf(gy, v, fAr);
            fAi = fmaf(gy, u, fAi); fAi = fmaf(-gx, v, fAi);
            fEr = fmaf(gz, u, fEr); fEr = fmaf(gw, v, fEr);
            fEi = fmaf(gw, u, fEi); fEi = fmaf(-gz, v, fEi);
        }
        acc.sAr += (double)fAr; acc.sAi += (double)fAi; acc.sEr += (double)fEr; acc.sEi += (double)fEi;
    }
}

// unmasked bins [b0, b1), b0 and b1 even: pairs of bins (2p, 2p+1) ride in the two lanes of f32x2 instructions
// (sin/cos polynomials, A e^{-i Psi}, MACs): fewer instructions, and none of the select / add bookkeeping of two
// scalar passes.  Each accumulator lane sums every other bin, so a flush every 2 kMixedChain bins keeps the chains
// at kMixedChain terms.  The four products g_re u, g_im v, g_im u, g_re v are summed separately (f32x2 FMA has no
// operand negation) and combined at the flush.
__device__ __forceinline__ void fused_pairs_mixed(int b0, int b1, int kbase, double df, double nxj, double cA0, double cA1,
                                                  double cA2, double cA3, double cP0, double cP1, double cP2, double cP3,
                                                  const float *__restrict__ sgp, const double *__restrict__ sWc,
                                                  MixedAcc &acc)
{
    for (int base = b0; base < b1; base += 2 * kMixedChain) {
        const int end = min(base + 2 * kMixedChain, b1);
        f32x2 aXU = 0, aYV = 0, aYU = 0, aXV = 0, eXU = 0, eYV = 0, eYU = 0, eXV = 0; // +0.0f in both lanes
#pragma unroll 2
        for (int ii = base; ii < end; ii += 2) {
            const double t0 = fma((double)(kbase + ii), df, nxj), t1 = fma((double)(kbase + ii + 1), df, nxj);
            const double A0 = fma(fma(fma(cA3, t0, cA2), t0, cA1), t0, cA0);
            const double A1 = fma(fma(fma(cA3, t1, cA2), t1, cA1), t1, cA0);
            const double y0 = fma(fma(fma(cP3, t0, cP2), t0, cP1), t0, cP0);
            const double y1 = fma(fma(fma(cP3, t1, cP2), t1, cP1), t1, cP0);
            const double2 w = *reinterpret_cast<const double2 *>(sWc + ii);
            acc.sH = fma(w.x * A0, A0, acc.sH);
            acc.sH = fma(w.y * A1, A1, acc.sH);
            int q0, q1;
            const float x0 = reduce_qc_to_rad_f32(y0, q0), x1 = reduce_qc_to_rad_f32(y1, q1);
            f32x2 S, C;
            sincos_poly_f32x2(pack2(x0, x1), S, C);
            float s0, s1, c0, c1, as0, as1, a0, a1, bb0, bb1;
            unpack2(S, s0, s1);
            unpack2(C, c0, c1);
            quadrant_f32(q0, __double2float_rn(A0), s0, c0, as0, a0, bb0);
            quadrant_f32(q1, __double2float_rn(A1), s1, c1, as1, a1, bb1);
            const f32x2 AS = pack2(as0, as1);
            const f32x2 U = mul2(AS, pack2(bb0, bb1)), V = mul2(AS, pack2(a0, a1)); // h = u - i v per lane
            const ulonglong2 gA = *reinterpret_cast<const ulonglong2 *>(sgp + (ii >> 1) * 8);
            const ulonglong2 gE = *reinterpret_cast<const ulonglong2 *>(sgp + (ii >> 1) * 8 + 4);
            aXU = fma2(gA.x, U, aXU); aYV = fma2(gA.y, V, aYV); aYU = fma2(gA.y, U, aYU); aXV = fma2(gA.x, V, aXV);
            eXU = fma2(gE.x, U, eXU); eYV = fma2(gE.y, V, eYV); eYU = fma2(gE.y, U, eYU); eXV = fma2(gE.x, V, eXV);
        }
        float l0, h0, l1, h1;
        // S^A_re = sum g_re u + g_im v,  S^A_im = sum g_im u - g_re v   (g already holds W conj(d))
        unpack2(aXU, l0, h0); unpack2(aYV, l1, h1); acc.sAr += (double)((l0 + h0) + (l1 + h1));
        unpack2(aYU, l0, h0); unpack2(aXV, l1, h1); acc.sAi += (double)((l0 + h0) - (l1 + h1));
        unpack2(eXU, l0, h0); unpack2(eYV, l1, h1); acc.sEr += (double)((l0 + h0) + (l1 + h1));
        unpack2(eYU, l0, h0); unpack2(eXV, l1, h1); acc.sEi += (double)((l0 + h0) - (l1 + h1));
    }
}

struct FusedArgsF32 {
    const float *g4f;   // [n_f_pad][4] binary32, g / sigma
    const double *Wds;  // [n_f_pad] FP64, W / sigma^2
    const double *scale;
};

__global__ void __launch_bounds__(128, 4) k_full_fused_mixed(FusedArgs a, FusedArgsF32 m)
{
    extern __shared__ __align__(128) double sm[];
    __shared__ __align__(8) uint64_t bar[2];
    __shared__ int s_lo, s_hi;

    const int tid = threadIdx.x;
    const int p = blockIdx.x * blockDim.x + tid;
    const int tile = blockIdx.y;
    const int i0 = __ldg(a.tile_start + tile), i1 = __ldg(a.tile_start + tile + 1); // tile = dense bins [i0, i1)
    const int lo = max(a.ilo[p], i0), hi = min(a.ihi[p], i1);
    if (tid == 0) {
        s_lo = INT_MAX;
        s_hi = INT_MIN;
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (lo < hi) {
        atomicMin(&s_lo, lo);
        atomicMax(&s_hi, hi);
    }
    __syncthreads();
    const int blo = s_lo, bhi = s_hi;
    if (blo >= bhi) return;

    const int CH = a.CH;
    const int c_begin = blo / CH, c_end = (bhi + CH - 1) / CH;
    // stage = CH float4 (g) + CH double (W) = 24 B per bin = 3 doubles
    const uint32_t stage_bytes = (uint32_t)CH * 24u;
    auto issue = [&](int c, int st) {
        double *dst = sm + (size_t)st * CH * 3;
        mbar_expect_tx(&bar[st], stage_bytes);
        tma_load_1d(dst, m.g4f + (size_t)c * CH * 4, (uint32_t)CH * 16u, &bar[st]);
        tma_load_1d(dst + (size_t)CH * 2, m.Wds + (size_t)c * CH, (uint32_t)CH * 8u, &bar[st]);
    };
    if (tid == 0) issue(c_begin, 0);

    const size_t sw = (size_t)a.n_wp;
    const size_t cj = (size_t)8 * sw;
    const double sigma = m.scale[0];
    const int kbase = (int)a.k_min;
    int j = find_interval_of_bin(a.bstart, a.n_nodes, blo);
    int jl = -1;
    double cA0 = 0, cA1 = 0, cA2 = 0, cA3 = 0, cP0 = 0, cP1 = 0, cP2 = 0, cP3 = 0, nxj = 0;
    MixedAcc acc{0, 0, 0, 0, 0};

    for (int c = c_begin; c < c_end; ++c) {
        const int st = (c - c_begin) & 1;
        const uint32_t ph = (uint32_t)((c - c_begin) >> 1) & 1u;
        if (tid == 0 && c + 1 < c_end) issue(c + 1, st ^ 1);
        mbar_wait(&bar[st], ph);
        const double *sg = sm + (size_t)st * CH * 3;
        const double *sW = sg + (size_t)CH * 2;
        const int cb = c * CH;
        const int ce = min(cb + CH, bhi);
        int i = max(cb, blo);
        while (i < ce) {
            while (j < a.n_nodes - 2 && __ldg(a.bstart + j + 1) <= i) ++j;
            const int seg_end = (j < a.n_nodes - 2) ? min(__ldg(a.bstart + j + 1), ce) : ce;
            int tlo = max(i, lo), thi = min(seg_end, hi);
            if (tlo >= thi) { tlo = INT_MAX; thi = INT_MIN; }
            const int wlo = __reduce_min_sync(0xffffffffu, tlo);
            const int whi = __reduce_max_sync(0xffffffffu, thi);
            if (wlo < whi) {
                if (j != jl) {
                    const double *cc = a.C + (size_t)j * cj + p;
                    cA0 = cc[0] * sigma; cA1 = cc[sw] * sigma; cA2 = cc[2 * sw] * sigma; cA3 = cc[3 * sw] * sigma;
                    cP0 = cc[4 * sw]; cP1 = cc[5 * sw]; cP2 = cc[6 * sw]; cP3 = cc[7 * sw];
                    nxj = -__ldg(a.xj + j);
                    jl = j;
                }
                const int flo = __reduce_max_sync(0xffffffffu, max(lo, i));
                const int fhi = __reduce_min_sync(0xffffffffu, min(hi, seg_end));
                const float *sgp = reinterpret_cast<const float *>(sg) - (size_t)cb * 4; // cb is even
                const double *sWc = sW - cb;
                // masked bins up to the first even bin every lane has, packed pairs, masked rest
                const int plo = (flo + 1) & ~1, phi = fhi & ~1;
                if (plo < phi) {
                    fused_bins_mixed<true>(wlo, plo, tlo, thi, kbase, a.df, nxj, cA0, cA1, cA2, cA3, cP0, cP1,
                                           cP2, cP3, sgp, sWc, acc);
                    fused_pairs_mixed(plo, phi, kbase, a.df, nxj, cA0, cA1, cA2, cA3, cP0, cP1, cP2, cP3, sgp, sWc, acc);
                    fused_bins_mixed<true>(phi, whi, tlo, thi, kbase, a.df, nxj, cA0, cA1, cA2, cA3, cP0, cP1,
                                           cP2, cP3, sgp, sWc, acc);
                } else {
                    fused_bins_mixed<true>(wlo, whi, tlo, thi, kbase, a.df, nxj, cA0, cA1, cA2, cA3, cP0, cP1,
                                           cP2, cP3, sgp, sWc, acc);
                }
            }
            i = seg_end;
        }
        __syncthreads();
    }
    double *o = a.part + ((size_t)tile * 5) * sw + p;
    o[0] = acc.sAr; o[sw] = acc.sAi; o[2 * sw] = acc.sEr; o[3 * sw] = acc.sEi; o[4 * sw] = acc.sH;
}

// ---------------------------------------------------------------------------------------------------
// F3 with a frequency-dependent transfer function (Eq. 8-9).  Same mapping, staging and
// band logic as k_full_fused; per (walker, bin, mode) six cubics (amplitude, phase, Re/Im of T^A and T^E), then
// h^c += T^c(f) A e^{-i Psi}.  Coefficient block per (interval, mode): 24 doubles, walker fastest.
// NM1 = 1: the 24 coefficients of the current interval live in registers; 0: any n_m, coefficients re-read per
// bin through L1 (they would not fit in registers for several modes).
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ double cubic4(const double *c4, double t)
{
    return fma(fma(fma(c4[3], t, c4[2]), t, c4[1]), t, c4[0]);
}

template <int NM1>
__global__ void __launch_bounds__(128, 3) k_full_fused_tf(FusedArgs a)
{
    extern __shared__ __align__(128) double sm[];
    __shared__ __align__(8) uint64_t bar[2];
    __shared__ int s_lo, s_hi;

    const int tid = threadIdx.x;
    const int p = blockIdx.x * blockDim.x + tid;
    const int tile = blockIdx.y;
    const int i0 = __ldg(a.tile_start + tile), i1 = __ldg(a.tile_start + tile + 1); // tile = dense bins [i0, i1)
    const int lo = max(a.ilo[p], i0), hi = min(a.ihi[p], i1);
    if (tid == 0) {
        s_lo = INT_MAX;
        s_hi = INT_MIN;
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (lo < hi) {
        atomicMin(&s_lo, lo);
        atomicMax(&s_hi, hi);
    }
    __syncthreads();
    const int blo = s_lo, bhi = s_hi;
    if (blo >= bhi) return;

    const int CH = a.CH;
    const int c_begin = blo / CH, c_end = (bhi + CH - 1) / CH;
    const uint32_t stage_bytes = (uint32_t)CH * 40u;
    auto issue = [&](int c, int st) {
        double *dst = sm + (size_t)st * CH * 5;
        mbar_expect_tx(&bar[st], stage_bytes);
        tma_load_1d(dst, a.g4 + (size_t)c * CH * 4, (uint32_t)CH * 32u, &bar[st]);
        tma_load_1d(dst + (size_t)CH * 4, a.Wd + (size_t)c * CH, (uint32_t)CH * 8u, &bar[st]);
    };
    if (tid == 0) issue(c_begin, 0);

    const size_t sw = (size_t)a.n_wp;
    const size_t cm = (size_t)24 * sw;          // one mode's block
    const size_t cj = (size_t)a.n_m * cm;       // one interval's block
    const int kbase = (int)a.k_min;
    int j = find_interval_of_bin(a.bstart, a.n_nodes, blo);
    int jl = -1;
    double co[24];
    double nxj = 0.0, s_dh = 0.0, s_hh = 0.0;

    for (int c = c_begin; c < c_end; ++c) {
        const int st = (c - c_begin) & 1;
        const uint32_t ph = (uint32_t)((c - c_begin) >> 1) & 1u;
        if (tid == 0 && c + 1 < c_end) issue(c + 1, st ^ 1);
        mbar_wait(&bar[st], ph);
        const double *sg = sm + (size_t)st * CH * 5;
        const double *sW = sg + (size_t)CH * 4;
        const int cb = c * CH;
        const int ce = min(cb + CH, bhi);
        int i = max(cb, blo);
        while (i < ce) {
            while (j < a.n_nodes - 2 && __ldg(a.bstart + j + 1) <= i) ++j;
            const int seg_end = (j < a.n_nodes - 2) ? min(__ldg(a.bstart + j + 1), ce) : ce;
            int tlo = max(i, lo), thi = min(seg_end, hi);
            if (tlo >= thi) { tlo = INT_MAX; thi = INT_MIN; }
            const int wlo = __reduce_min_sync(0xffffffffu, tlo);
            const int whi = __reduce_max_sync(0xffffffffu, thi);
            if (wlo < whi) {
                const double *cc0 = a.C + (size_t)j * cj + p;
                if (j != jl) {
                    nxj = -__ldg(a.xj + j);
                    if (NM1) {
#pragma unroll
                        for (int q = 0; q < 24; ++q) co[q] = cc0[(size_t)q * sw];
                    }
                    jl = j;
                }
                const double4 *sg4 = reinterpret_cast<const double4 *>(sg) - cb;
                const double *sWc = sW - cb;
                auto direct_bins = [&](int b0, int b1) {
                    if (!NM1) {
                        // several modes: chunks of four bins, mode loop outside (24 coefficients read once per chunk)
                        for (int c4 = b0; c4 < b1; c4 += 4) {
                            double t4[4], h4[4][4];
#pragma unroll
                            for (int k = 0; k < 4; ++k) {
                                t4[k] = fma((double)(kbase + c4 + k), a.df, nxj);
                                h4[k][0] = h4[k][1] = h4[k][2] = h4[k][3] = 0.0;
                            }
#pragma unroll 1
                            for (int m = 0; m < a.n_m; ++m) {
                                const double *cc = cc0 + (size_t)m * cm;
#pragma unroll
                                for (int q = 0; q < 24; ++q) co[q] = cc[(size_t)q * sw];
#pragma unroll
                                for (int k = 0; k < 4; ++k) {
                                    const double t = t4[k];
                                    const double A = cubic4(co, t), y = cubic4(co + 4, t);
                                    const double tar = cubic4(co + 8, t), tai = cubic4(co + 12, t);
                                    const double ter = cubic4(co + 16, t), tei = cubic4(co + 20, t);
                                    double u, v; // h_m = u - i v
                                    amp_expi_qc(A, y, u, v);
                                    h4[k][0] = fma(tar, u, h4[k][0]); h4[k][0] = fma(tai, v, h4[k][0]);
                                    h4[k][1] = fma(tai, u, h4[k][1]); h4[k][1] = fma(-tar, v, h4[k][1]);
                                    h4[k][2] = fma(ter, u, h4[k][2]); h4[k][2] = fma(tei, v, h4[k][2]);
                                    h4[k][3] = fma(tei, u, h4[k][3]); h4[k][3] = fma(-ter, v, h4[k][3]);
                                }
                            }
#pragma unroll
                            for (int k = 0; k < 4; ++k) {
                                const int ii = c4 + k;
                                if (ii < b1 && ii >= tlo && ii < thi) {
                                    const double4 g = sg4[ii];
                                    const double w = sWc[ii];
                                    s_dh = fma(g.x, h4[k][0], s_dh); s_dh = fma(-g.y, h4[k][1], s_dh);
                                    s_dh = fma(g.z, h4[k][2], s_dh); s_dh = fma(-g.w, h4[k][3], s_dh);
                                    s_hh = fma(w, fma(h4[k][0], h4[k][0], h4[k][1] * h4[k][1]) +
                                                      fma(h4[k][2], h4[k][2], h4[k][3] * h4[k][3]), s_hh);
                                }
                            }
                        }
                        return;
                    }
#pragma unroll 2
                    for (int ii = b0; ii < b1; ++ii) {
                        const bool act = (ii >= tlo) && (ii < thi);
                        const double t = fma((double)(kbase + ii), a.df, nxj);
                        double hAr = 0, hAi = 0, hEr = 0, hEi = 0;
                        const int n_m = NM1 ? 1 : a.n_m;
                        for (int m = 0; m < n_m; ++m) {
                            if (!NM1) {
                                const double *cc = cc0 + (size_t)m * cm;
#pragma unroll
                                for (int q = 0; q < 24; ++q) co[q] = cc[(size_t)q * sw];
                            }
                            const double A = cubic4(co, t), y = cubic4(co + 4, t);
                            const double tar = cubic4(co + 8, t), tai = cubic4(co + 12, t);
                            const double ter = cubic4(co + 16, t), tei = cubic4(co + 20, t);
                            double u, v; // h_m = u - i v
                            amp_expi_qc(A, y, u, v);
                            hAr = fma(tar, u, hAr); hAr = fma(tai, v, hAr);
                            hAi = fma(tai, u, hAi); hAi = fma(-tar, v, hAi);
                            hEr = fma(ter, u, hEr); hEr = fma(tei, v, hEr);
                            hEi = fma(tei, u, hEi); hEi = fma(-ter, v, hEi);
                        }
                        if (act) {
                            const double4 g = sg4[ii];
                            const double w = sWc[ii];
                            s_dh = fma(g.x, hAr, s_dh); s_dh = fma(-g.y, hAi, s_dh);
                            s_dh = fma(g.z, hEr, s_dh); s_dh = fma(-g.w, hEi, s_dh);
                            s_hh = fma(w, fma(hAr, hAr, hAi * hAi) + fma(hEr, hEr, hEi * hEi), s_hh);
                        }
                    }
                };
                // bins inside every lane's band: e^{-i Psi} and A by the recurrence of fused_bins_rot, T^c(f) by Horner
                const int flo = __reduce_max_sync(0xffffffffu, max(lo, i));
                const int fhi = __reduce_min_sync(0xffffffffu, min(hi, seg_end));
                if (NM1 && LL_FUSED_ROT && fhi - flo >= 8) {
                    direct_bins(wlo, flo);
                    const double df = a.df, df2 = df * df, df3 = df2 * df;
                    const double d3A = 6.0 * co[3] * df3;
                    double su, cu;
                    sincos_qc(6.0 * co[7] * df3, su, cu);
                    unit_modulus(cu, su);
                    for (int k0 = flo; k0 < fhi; k0 += kRotSync) {
                        const int k1 = min(k0 + kRotSync, fhi);
                        const double t0 = fma((double)(kbase + k0), df, nxj);
                        const double tt = fma(2.0, t0, df), q3 = fma(3.0 * t0, t0 + df, df2), t1 = t0 + df;
                        double A = cubic4(co, t0);
                        double d1A = df * fma(co[3], q3, fma(co[2], tt, co[1]));
                        double d2A = df2 * fma(6.0 * co[3], t1, 2.0 * co[2]);
                        double sz, cz, sw_, cw, sv, cv;
                        sincos_qc(cubic4(co + 4, t0), sz, cz);
                        sincos_qc(df * fma(co[7], q3, fma(co[6], tt, co[5])), sw_, cw);
                        sincos_qc(df2 * fma(6.0 * co[7], t1, 2.0 * co[6]), sv, cv);
                        unit_modulus(cz, sz); unit_modulus(cw, sw_); unit_modulus(cv, sv);
#pragma unroll 2
                        for (int ii = k0; ii < k1; ++ii) {
                            const double t = fma((double)(kbase + ii), df, nxj);
                            const double tar = cubic4(co + 8, t), tai = cubic4(co + 12, t);
                            const double ter = cubic4(co + 16, t), tei = cubic4(co + 20, t);
                            const double u = A * cz, v = A * sz; // h = u - i v
                            const double hAr = fma(tar, u, tai * v), hAi = fma(tai, u, -(tar * v));
                            const double hEr = fma(ter, u, tei * v), hEi = fma(tei, u, -(ter * v));
                            const double4 g = sg4[ii];
                            const double w = sWc[ii];
                            s_dh = fma(g.x, hAr, s_dh); s_dh = fma(-g.y, hAi, s_dh);
                            s_dh = fma(g.z, hEr, s_dh); s_dh = fma(-g.w, hEi, s_dh);
                            s_hh = fma(w, fma(hAr, hAr, hAi * hAi) + fma(hEr, hEr, hEi * hEi), s_hh);
                            const double nzc = fma(cz, cw, -(sz * sw_)), nzs = fma(sz, cw, cz * sw_);
                            const double nwc = fma(cw, cv, -(sw_ * sv)), nws = fma(sw_, cv, cw * sv);
                            const double nvc = fma(cv, cu, -(sv * su)), nvs = fma(sv, cu, cv * su);
                            cz = nzc; sz = nzs; cw = nwc; sw_ = nws; cv = nvc; sv = nvs;
                            A += d1A; d1A += d2A; d2A += d3A;
                        }
                    }
                    direct_bins(fhi, whi);
                } else {
                    direct_bins(wlo, whi);
                }
            }
            i = seg_end;
        }
        __syncthreads();
    }
    double *o = a.part + ((size_t)tile * 2) * sw + p;
    o[0] = s_dh; o[sw] = s_hh;
}

// ---------------------------------------------------------------------------------------------------
// Per-walker node grids (reading R30): every walker has its own nodes x_{w,j}, hence its own
// tridiagonal matrix (a true batched solve) and its own bin -> interval map.
// ---------------------------------------------------------------------------------------------------
// X[j][p] = f_nodes_w[perm[p]][j] (walker fastest); padding positions get an ascending dummy grid.
// band_w[w] = [max(band_lo, x_0), min(band_hi, x_last)]: a spline is not extrapolated beyond its own nodes.
__global__ void __launch_bounds__(256)
k_pw_band(const double *__restrict__ f_nodes_w, const double *__restrict__ band, int n_w, int n_nodes,
          double *__restrict__ band_w)
{
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= n_w) return;
    double lo = f_nodes_w[(size_t)w * n_nodes], hi = f_nodes_w[(size_t)w * n_nodes + n_nodes - 1];
    if (band) { lo = fmax(lo, band[2 * (size_t)w]); hi = fmin(hi, band[2 * (size_t)w + 1]); }
    band_w[2 * (size_t)w] = lo;
    band_w[2 * (size_t)w + 1] = hi;
}

__global__ void __launch_bounds__(256)
k_pw_nodes_x(const double *__restrict__ f_nodes_w, const int *__restrict__ perm, int n_wp, int n_nodes, double *__restrict__ X)
{
    __shared__ double tt[32][33];
    const int p0 = blockIdx.x * 32, j0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5; // 32 x 8
    for (int r = ty; r < 32; r += 8) {
        const int w = perm[p0 + r];
        const int j = j0 + tx;
        tt[r][tx] = (j < n_nodes) ? (w >= 0 ? f_nodes_w[(size_t)w * n_nodes + j] : (double)(j + 1)) : 0.0;
    }
    __syncthreads();
    for (int r = ty; r < 32; r += 8) {
        const int j = j0 + r;
        if (j < n_nodes) X[(size_t)j * n_wp + p0 + tx] = tt[tx][r];
    }
}

// F2, one thread per system, full Thomas elimination with the walker's own nodes (reading R1: natural BC).
// c'_j and dp_j are parked in the c- and b-slots of interval j between the sweeps.
__global__ void __launch_bounds__(128)
k_spline_pw(const double *__restrict__ Y, const double *__restrict__ X, double *__restrict__ C, int n_wp, int n_nodes, int n_m,
            int bc)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_wp) return;
    const int sys = blockIdx.y, m = sys >> 1, kind = sys & 1;
    const size_t sw = (size_t)n_wp;
    const double *y = Y + (size_t)sys * n_nodes * sw + p;
    const double *x = X + p;
    double *c = C + ((size_t)m * 8 + kind * 4) * sw + p;
    const size_t cj = (size_t)n_m * 8 * sw;
    const int n = n_nodes;
    double x0 = __ldg(x), x1 = __ldg(x + sw), y0 = __ldg(y), y1 = __ldg(y + sw);
    double hm = x1 - x0, sprev = (y1 - y0) / hm;
    double cpp = 0.0, dpp = 0.0, rho0 = 0.0, rhon = 0.0;
#pragma unroll 4
    for (int j = 1; j <= n - 2; ++j) {
        const double x2 = __ldg(x + (size_t)(j + 1) * sw), y2 = __ldg(y + (size_t)(j + 1) * sw);
        const double hp = x2 - x1;
        const double s = (y2 - y1) / hp;
        double a = hm * kSixth, b = (hm + hp) * (1.0 / 3.0), cc = hp * kSixth;
        if (bc) { // not-a-knot: end conditions substituted into rows 1 and n-2
            if (j == 1) { rho0 = hm / hp; b += a * (1.0 + rho0); cc -= a * rho0; }
            if (j == n - 2) { rhon = hp / hm; b += cc * (1.0 + rhon); a -= cc * rhon; cc = 0.0; }
        }
        if (j == 1) a = 0.0;
        const double inv = 1.0 / (b - a * cpp);
        const double cp = cc * inv, dp = ((s - sprev) - a * dpp) * inv;
        c[(size_t)j * cj + sw] = dp;
        c[(size_t)j * cj + 2 * sw] = cp;
        cpp = cp; dpp = dp; sprev = s; hm = hp; x1 = x2; y1 = y2;
    }
    double Mn = 0.0, Mnn = 0.0;
    if (bc) {
        const double M2 = c[(size_t)(n - 2) * cj + sw];
        const double M3 = fma(-c[(size_t)(n - 3) * cj + 2 * sw], M2, c[(size_t)(n - 3) * cj + sw]);
        Mn = (1.0 + rhon) * M2 - rhon * M3;
    }
    double xh = __ldg(x + (size_t)(n - 1) * sw), yh = __ldg(y + (size_t)(n - 1) * sw);
    // backward sweep in register blocks of 8 rows (loads first, then the recurrence, then the stores): a load of the
    // parked c', dp of row j issued between the stores of row j + 1 could not be hoisted (same base pointer)
    constexpr int kB = 8;
    for (int jt = n - 2; jt >= 0; jt -= kB) {
        double xv[kB], yv[kB], dpv[kB], cpv[kB];
#pragma unroll
        for (int k = 0; k < kB; ++k) {
            const int j = jt - k;
            xv[k] = (j >= 0) ? __ldg(x + (size_t)j * sw) : 0.0;
            yv[k] = (j >= 0) ? __ldg(y + (size_t)j * sw) : 0.0;
            dpv[k] = (j >= 1) ? c[(size_t)j * cj + sw] : 0.0;
            cpv[k] = (j >= 1) ? c[(size_t)j * cj + 2 * sw] : 0.0;
        }
#pragma unroll
        for (int k = 0; k < kB; ++k) {
            const int j = jt - k;
            if (j >= 0) {
                const double xl = xv[k], yl = yv[k];
                double *cc = c + (size_t)j * cj;
                const double Mj = (j >= 1) ? fma(-cpv[k], Mn, dpv[k]) : (bc ? (1.0 + rho0) * Mn - rho0 * Mnn : 0.0);
                const double h = xh - xl, ih = 1.0 / h;
                cc[0] = yl;
                cc[sw] = (yh - yl) * ih - h * (2.0 * Mj + Mn) * kSixth;
                cc[2 * sw] = 0.5 * Mj;
                cc[3 * sw] = (Mn - Mj) * ih * kSixth;
                Mnn = Mn; Mn = Mj; xh = xl; yh = yl;
            }
        }
    }
}

// F3 with per-walker intervals.  Same mapping and data staging as k_full_fused_tf (one thread = one walker, TMA-fed
// g/W tiles broadcast from shared memory); every lane tracks its own interval: the bins go up, so the interval index
// only moves forward, by a comparison with the lane's next node per bin.  NM1: the 8 coefficients of the lane's
// current interval live in registers; otherwise they are re-read per bin through L1.
template <int NM1>
__global__ void __launch_bounds__(128, 3) k_full_fused_pw(FusedArgs a, const double *__restrict__ X)
{
    extern __shared__ __align__(128) double sm[];
    __shared__ __align__(8) uint64_t bar[2];
    __shared__ int s_lo, s_hi;

    const int tid = threadIdx.x;
    const int p = blockIdx.x * blockDim.x + tid;
    const int tile = blockIdx.y;
    const int i0 = __ldg(a.tile_start + tile), i1 = __ldg(a.tile_start + tile + 1);
    const int lo = max(a.ilo[p], i0), hi = min(a.ihi[p], i1);
    if (tid == 0) {
        s_lo = INT_MAX;
        s_hi = INT_MIN;
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (lo < hi) {
        atomicMin(&s_lo, lo);
        atomicMax(&s_hi, hi);
    }
    __syncthreads();
    const int blo = s_lo, bhi = s_hi;
    if (blo >= bhi) return;

    const int CH = a.CH;
    const int c_begin = blo / CH, c_end = (bhi + CH - 1) / CH;
    const uint32_t stage_bytes = (uint32_t)CH * 40u;
    auto issue = [&](int c, int st) {
        double *dst = sm + (size_t)st * CH * 5;
        mbar_expect_tx(&bar[st], stage_bytes);
        tma_load_1d(dst, a.g4 + (size_t)c * CH * 4, (uint32_t)CH * 32u, &bar[st]);
        tma_load_1d(dst + (size_t)CH * 4, a.Wd + (size_t)c * CH, (uint32_t)CH * 8u, &bar[st]);
    };
    if (tid == 0) issue(c_begin, 0);

    const size_t sw = (size_t)a.n_wp;
    const size_t cm = (size_t)8 * sw, cj = (size_t)a.n_m * cm;
    const int n = a.n_nodes;
    const double *x = X + p;
    // this lane's interval at its first bin: largest j in [0, n-2] with x_j <= f
    int j = 0;
    double xj = 0.0, xnext = INFINITY;
    double co[8];
    auto load_interval = [&](int jj) {
        xj = __ldg(x + (size_t)jj * sw);
        xnext = (jj < n - 2) ? __ldg(x + (size_t)(jj + 1) * sw) : INFINITY;
        if (NM1) {
            const double *cc = a.C + (size_t)jj * cj + p;
#pragma unroll
            for (int q = 0; q < 8; ++q) co[q] = cc[(size_t)q * sw];
        }
    };
    if (lo < hi) {
        const double f0 = (double)(a.k_min + lo) * a.df;
        int l = 0, h = n - 2;
        while (l < h) {
            const int mid = (l + h + 1) >> 1;
            if (__ldg(x + (size_t)mid * sw) <= f0) l = mid; else h = mid - 1;
        }
        j = l;
        load_interval(j);
    }
    double tf1[4] = {0, 0, 0, 0}; // single mode: the walker's transfer factors stay in registers
    if (NM1) { tf1[0] = a.TF[p]; tf1[1] = a.TF[sw + p]; tf1[2] = a.TF[2 * sw + p]; tf1[3] = a.TF[3 * sw + p]; }
    double s_dh = 0.0, s_hh = 0.0;

    for (int c = c_begin; c < c_end; ++c) {
        const int st = (c - c_begin) & 1;
        const uint32_t ph = (uint32_t)((c - c_begin) >> 1) & 1u;
        if (tid == 0 && c + 1 < c_end) issue(c + 1, st ^ 1);
        mbar_wait(&bar[st], ph);
        const double *sg = sm + (size_t)st * CH * 5;
        const double *sW = sg + (size_t)CH * 4;
        const int cb = c * CH;
        const int tlo = max(cb, lo), thi = min(cb + CH, hi);
        const double4 *sg4 = reinterpret_cast<const double4 *>(sg) - cb;
        const double *sWc = sW - cb;
        auto one_bin = [&](int ii, double f) {
            const double t = f - xj;
            double hAr = 0, hAi = 0, hEr = 0, hEi = 0;
            const int n_m = NM1 ? 1 : a.n_m;
            for (int m = 0; m < n_m; ++m) {
                if (!NM1) {
                    const double *cc = a.C + (size_t)j * cj + (size_t)m * cm + p;
#pragma unroll
                    for (int q = 0; q < 8; ++q) co[q] = cc[(size_t)q * sw];
                }
                const double A = cubic4(co, t), y = cubic4(co + 4, t);
                double u, v; // h_m = u - i v
                amp_expi_qc(A, y, u, v);
                double tar = tf1[0], tai = tf1[1], ter = tf1[2], tei = tf1[3];
                if (!NM1) {
                    const double *tf = a.TF + (size_t)m * 4 * sw + p;
                    tar = tf[0]; tai = tf[sw]; ter = tf[2 * sw]; tei = tf[3 * sw];
                }
                hAr = fma(tar, u, hAr); hAr = fma(tai, v, hAr);
                hAi = fma(tai, u, hAi); hAi = fma(-tar, v, hAi);
                hEr = fma(ter, u, hEr); hEr = fma(tei, v, hEr);
                hEi = fma(tei, u, hEi); hEi = fma(-ter, v, hEi);
            }
            const double4 g = sg4[ii];
            const double w = sWc[ii];
            s_dh = fma(g.x, hAr, s_dh); s_dh = fma(-g.y, hAi, s_dh);
            s_dh = fma(g.z, hEr, s_dh); s_dh = fma(-g.w, hEi, s_dh);
            s_hh = fma(w, fma(hAr, hAr, hAi * hAi) + fma(hEr, hEr, hEi * hEi), s_hh);
        };
        int ii = tlo;
        while (ii < thi) {
            const double f = (double)(a.k_min + ii) * a.df;
            while (f >= xnext) load_interval(++j);
            // while the next bins stay inside this lane's interval (intervals are hundreds of bins wide almost
            // everywhere) they go by the recurrence route of fused_bins_rot: up to kRotSync bins per re-sync
            int m = 0;
            if (NM1 && LL_FUSED_ROT) {
                m = min(thi - ii, kRotSync);
                const double room = (xnext - f) / a.df; // bins ii .. ii + ceil(room) - 1 lie below the next node
                if (room < (double)m) m = (int)room;    // conservative: the bin at the boundary takes the exact route
            }
            if (m >= 8) {
                const double df = a.df, df2 = df * df, df3 = df2 * df;
                const double t = f - xj, tt = fma(2.0, t, df), q3 = fma(3.0 * t, t + df, df2), t1 = t + df;
                double A = cubic4(co, t);
                double d1A = df * fma(co[3], q3, fma(co[2], tt, co[1]));
                double d2A = df2 * fma(6.0 * co[3], t1, 2.0 * co[2]);
                const double d3A = 6.0 * co[3] * df3;
                double sz, cz, sw_, cw, sv, cv, su, cu;
                sincos_qc(cubic4(co + 4, t), sz, cz);
                sincos_qc(df * fma(co[7], q3, fma(co[6], tt, co[5])), sw_, cw);
                sincos_qc(df2 * fma(6.0 * co[7], t1, 2.0 * co[6]), sv, cv);
                sincos_qc(6.0 * co[7] * df3, su, cu);
                unit_modulus(cz, sz); unit_modulus(cw, sw_); unit_modulus(cv, sv); unit_modulus(cu, su);
#pragma unroll 2
                for (int k = 0; k < m; ++k) {
                    const double u = A * cz, v = A * sz; // h = u - i v
                    const double hAr = fma(tf1[0], u, tf1[1] * v), hAi = fma(tf1[1], u, -(tf1[0] * v));
                    const double hEr = fma(tf1[2], u, tf1[3] * v), hEi = fma(tf1[3], u, -(tf1[2] * v));
                    const double4 g = sg4[ii + k];
                    const double w = sWc[ii + k];
                    s_dh = fma(g.x, hAr, s_dh); s_dh = fma(-g.y, hAi, s_dh);
                    s_dh = fma(g.z, hEr, s_dh); s_dh = fma(-g.w, hEi, s_dh);
                    s_hh = fma(w, fma(hAr, hAr, hAi * hAi) + fma(hEr, hEr, hEi * hEi), s_hh);
                    const double nzc = fma(cz, cw, -(sz * sw_)), nzs = fma(sz, cw, cz * sw_);
                    const double nwc = fma(cw, cv, -(sw_ * sv)), nws = fma(sw_, cv, cw * sv);
                    const double nvc = fma(cv, cu, -(sv * su)), nvs = fma(sv, cu, cv * su);
                    cz = nzc; sz = nzs; cw = nwc; sw_ = nws; cv = nvc; sv = nvs;
                    A += d1A; d1A += d2A; d2A += d3A;
                }
                ii += m;
            } else {
                one_bin(ii, f);
                ii += 1;
            }
        }
        __syncthreads();
    }
    double *o = a.part + ((size_t)tile * 2) * sw + p;
    o[0] = s_dh; o[sw] = s_hh;
}

// Eq. 8 utility: t_lm(f_j) = t_ref - (1/2pi) dphi/df at the nodes, dphi/df from the natural spline of the caller's
// node phases [n_sys][n_nodes] (radians).  One thread per system (off the hot path: the caller needs t_lm to build
// T(f, t_lm(f)) at the nodes).  scratch [n_nodes][n_sys] holds the forward-sweep values.
__global__ void __launch_bounds__(128)
k_tlm_nodes(const double *__restrict__ phase, int n_sys, int n_nodes, double t_ref, NodeTables nt,
            double *__restrict__ scratch, double *__restrict__ t_lm)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n_sys) return;
    const double *y = phase + (size_t)s * n_nodes;
    double *out = t_lm + (size_t)s * n_nodes;
    const int n = n_nodes;
    double ycur = y[1], sprev = (y[1] - y[0]) * __ldg(nt.invh), dpp = 0.0;
    for (int j = 1; j <= n - 2; ++j) {
        const double ynext = y[j + 1];
        const double sl = (ynext - ycur) * __ldg(nt.invh + j);
        const double dp = ((sl - sprev) - __ldg(nt.ta + j) * dpp) * __ldg(nt.tinv + j);
        scratch[(size_t)j * n_sys + s] = dp;
        dpp = dp;
        sprev = sl;
        ycur = ynext;
    }
    const double inv2pi = 0.5 / kPi;
    double Mn = 0.0, y1 = y[n - 1];
    for (int j = n - 2; j >= 0; --j) {
        const double y0 = y[j];
        const double Mj = (j >= 1) ? fma(-__ldg(nt.tcp + j), Mn, scratch[(size_t)j * n_sys + s]) : 0.0;
        const double h = __ldg(nt.hj + j), ih = __ldg(nt.invh + j);
        const double sl = (y1 - y0) * ih;
        if (j == n - 2) out[n - 1] = t_ref - (sl + h * (Mj + 2.0 * Mn) * kSixth) * inv2pi; // right end of the last interval
        out[j] = t_ref - (sl - h * (2.0 * Mj + Mn) * kSixth) * inv2pi;
        Mn = Mj;
        y1 = y0;
    }
}

// F4, first stage for small batches with thousands of tiles: block (x, z) adds, for its 32 walkers, the partials of
// the tiles of chunk z = [z cs, (z+1) cs) that lie in the walker's band, in a fixed order, into part2[z][NQ][n_wp];
// k_finalize then runs over the chunks as if they were tiles (tile_start2[z] = tile_start[z cs]).
template <int NQ>
__global__ void __launch_bounds__(32 * 32)
k_reduce_tiles(const double *__restrict__ part, const int *__restrict__ ilo, const int *__restrict__ ihi, int n_wp,
               const int *__restrict__ tile_start, int n_tiles, int cs, double *__restrict__ part2)
{
    __shared__ double red[32][NQ][32];
    const int p = blockIdx.x * 32 + threadIdx.x, ty = threadIdx.y, z = blockIdx.y;
    const bool in = p < n_wp;
    const size_t sw = (size_t)n_wp;
    const int lo = in ? ilo[p] : 0, hi = in ? ihi[p] : 0;
    double acc[NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) acc[q] = 0.0;
    bool any = false;
    if (hi > lo) {
        const int t0 = max(tile_of_bin(tile_start, n_tiles, lo), z * cs);
        const int t1 = min(tile_of_bin(tile_start, n_tiles, hi - 1), min((z + 1) * cs, n_tiles) - 1);
        any = t0 <= t1;
        for (int t = t0 + ty; t <= t1; t += 32) {
            const double *o = part + ((size_t)t * NQ) * sw + p;
#pragma unroll
            for (int q = 0; q < NQ; ++q) acc[q] += o[q * sw];
        }
    }
#pragma unroll
    for (int q = 0; q < NQ; ++q) red[ty][q][threadIdx.x] = acc[q];
    __syncthreads();
    if (ty != 0 || !in || !any) return;
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        double v = red[0][q][threadIdx.x];
#pragma unroll
        for (int k = 1; k < 32; ++k) v += red[k][q][threadIdx.x];
        part2[((size_t)z * NQ + q) * sw + p] = v;
    }
}

// F4: reduce the per-tile partials in a fixed order, apply T^c (single mode), form log L        (Eq. 2)
// Block = 32 walkers x kFinY tile slices: slice ty sums tiles t0 + ty, t0 + ty + kFinY, ... of its walker, the
// slices meet in shared memory and are added in slice order (deterministic: reruns are bit-identical).
constexpr int kFinY = 32;
template <int NM1>
__global__ void __launch_bounds__(32 * kFinY)
k_finalize(const double *__restrict__ part, const double *__restrict__ TF, const int *__restrict__ perm,
           const int *__restrict__ ilo, const int *__restrict__ ihi, int n_wp, const int *__restrict__ tile_start,
           int n_tiles, const double *__restrict__ dd, double *__restrict__ logL, double *__restrict__ d_h,
           double *__restrict__ h_h)
{
    constexpr int NQ = NM1 ? 5 : 2;
    __shared__ double red[kFinY][NQ][32];
    const int p = blockIdx.x * 32 + threadIdx.x, ty = threadIdx.y;
    const bool in = p < n_wp;
    const size_t sw = (size_t)n_wp;
    const int lo = in ? ilo[p] : 0, hi = in ? ihi[p] : 0;
    double acc[NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) acc[q] = 0.0;
    if (hi > lo) {
        const int t0 = tile_of_bin(tile_start, n_tiles, lo), t1 = tile_of_bin(tile_start, n_tiles, hi - 1);
#pragma unroll 4
        for (int t = t0 + ty; t <= t1; t += kFinY) {
            const double *o = part + ((size_t)t * NQ) * sw + p;
#pragma unroll
            for (int q = 0; q < NQ; ++q) acc[q] += o[q * sw];
        }
    }
#pragma unroll
    for (int q = 0; q < NQ; ++q) red[ty][q][threadIdx.x] = acc[q];
    __syncthreads();
    if (ty != 0 || !in) return;
    const int w = perm[p];
    if (w < 0) return;
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        double v = red[0][q][threadIdx.x];
#pragma unroll
        for (int k = 1; k < kFinY; ++k) v += red[k][q][threadIdx.x];
        acc[q] = v;
    }
    double dh, hh;
    if (NM1) {
        const double tar = TF[p], tai = TF[sw + p], ter = TF[2 * sw + p], tei = TF[3 * sw + p];
        // Re[T^A S^A + T^E S^E],  (|T^A|^2 + |T^E|^2) H
        dh = (tar * acc[0] - tai * acc[1]) + (ter * acc[2] - tei * acc[3]);
        hh = (tar * tar + tai * tai + ter * ter + tei * tei) * acc[4];
    } else {
        dh = acc[0];
        hh = acc[1];
    }
    logL[w] = dh - 0.5 * hh - 0.5 * dd[0];
    if (d_h) d_h[w] = dh;
    if (h_h) h_h[w] = hh;
}

// dense template of the walker at sorted position p (setup utility; same arithmetic as k_full_fused)
__global__ void __launch_bounds__(256)
k_full_template(FusedArgs a, int p, double *__restrict__ h_out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.n_f) return;
    double hAr = 0, hAi = 0, hEr = 0, hEi = 0;
    if (i >= a.ilo[p] && i < a.ihi[p]) {
        const int j = find_interval_of_bin(a.bstart, a.n_nodes, (int)i);
        const size_t sw = (size_t)a.n_wp;
        const double t = fma((double)(a.k_min + i), a.df, -a.xj[j]);
        for (int m = 0; m < a.n_m; ++m) {
            const double *cc = a.C + ((size_t)j * a.n_m + m) * 8 * sw + p;
            const double A = fma(fma(fma(cc[3 * sw], t, cc[2 * sw]), t, cc[sw]), t, cc[0]);
            const double y = fma(fma(fma(cc[7 * sw], t, cc[6 * sw]), t, cc[5 * sw]), t, cc[4 * sw]);
            double sn, cs;
            sincos_qc(y, sn, cs);
            const double u = A * cs, v = A * sn;
            const double *tf = a.TF + (size_t)m * 4 * sw + p;
            const double tar = tf[0], tai = tf[sw], ter = tf[2 * sw], tei = tf[3 * sw];
            hAr = fma(tar, u, hAr); hAr = fma(tai, v, hAr);
            hAi = fma(tai, u, hAi); hAi = fma(-tar, v, hAi);
            hEr = fma(ter, u, hEr); hEr = fma(tei, v, hEr);
            hEi = fma(tei, u, hEi); hEi = fma(-ter, v, hEi);
        }
    }
    reinterpret_cast<double2 *>(h_out)[i] = make_double2(hAr, hAi);
    reinterpret_cast<double2 *>(h_out)[a.n_f + i] = make_double2(hEr, hEi);
}

// stand-in template of one parameter row evaluated directly at arbitrary frequencies (no spline, no tables)
struct DirectRow {
    double p[5 + 4 * kMaxModes];
    double c_lm[kMaxModes];
};
struct DirectClm {
    double c_lm[kMaxModes];
};

// h^A, h^E of one stand-in parameter row at frequency fi, evaluated directly (Eq. 7, 9; reading R9)
__device__ __forceinline__ void direct_template_at(const double *__restrict__ rp, const double *__restrict__ c_lm,
                                                   const StandinInfo &si, double Mtot, double eta, double fisco,
                                                   double fi, double &hAr, double &hAi, double &hEr, double &hEi)
{
    const double tc = rp[2], phic = rp[3], invD = rp[4];
    const double inv_kappa = 1.0 / si.kappa;
    hAr = hAi = hEr = hEi = 0.0;
    for (int m = 0; m < si.n_m; ++m) {
        const double mh = 0.5 * (double)si.mode_m[m];
        const double fp = fi / mh;
        const double A = c_lm[m] * pow(fi, -7.0 / 6.0) * invD * taper(fp / fisco, si.kappa, inv_kappa);
        const double v = cbrt(kPi * Mtot * fp);
        const double v2 = v * v;
        const double psi = mh * (2.0 * kPi * fp * tc - phic - 0.25 * kPi + 3.0 / (128.0 * eta * (v2 * v2 * v)));
        double sn, cs;
        sincos_rad(psi, sn, cs);
        const double u = A * cs, vv = A * sn;
        const double tar = rp[5 + m * 4], tai = rp[6 + m * 4], ter = rp[7 + m * 4], tei = rp[8 + m * 4];
        hAr = fma(tar, u, hAr); hAr = fma(tai, vv, hAr);
        hAi = fma(tai, u, hAi); hAi = fma(-tar, vv, hAi);
        hEr = fma(ter, u, hEr); hEr = fma(tei, vv, hEr);
        hEi = fma(tei, u, hEi); hEi = fma(-ter, vv, hEi);
    }
}

// f == NULL: the frequencies are the dense grid's own, f_i = (k_min + i) df
__global__ void __launch_bounds__(256)
k_template_direct(DirectRow row, StandinInfo si, long long n_freq, const double *__restrict__ f, GridInfo g, double f_lo,
                  double f_hi, double *__restrict__ h_out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_freq) return;
    const double fi = f ? f[i] : bin_freq(g.k_min, i, g.df);
    double hAr = 0, hAi = 0, hEr = 0, hEi = 0;
    if (fi >= f_lo && fi <= f_hi) {
        double Mtot, eta, fisco;
        standin_masses(row.p[0], row.p[1], Mtot, eta, fisco);
        direct_template_at(row.p, row.c_lm, si, Mtot, eta, fisco, fi, hAr, hAi, hEr, hEi);
    }
    reinterpret_cast<double2 *>(h_out)[i] = make_double2(hAr, hAi);
    reinterpret_cast<double2 *>(h_out)[n_freq + i] = make_double2(hEr, hEi);
}

// PAPER.md:210 "replacing it with the highest Likelihood point in the population": index of the largest finite
// log L (lowest index on ties), one block; out_idx = -1 when no entry is finite.
__global__ void __launch_bounds__(1024) k_argmax(const double *__restrict__ v, long long n, long long *__restrict__ out_idx)
{
    __shared__ double sv[32];
    __shared__ long long si_[32];
    double bv = -INFINITY;
    long long bi = -1;
    for (long long i = threadIdx.x; i < n; i += blockDim.x) {
        const double x = v[i];
        if (x == x && fabs(x) != INFINITY && (bi < 0 || x > bv)) { bv = x; bi = i; } // ascending i: ties keep the lowest
    }
    auto better = [](double xv, long long xi, double yv, long long yi) {
        if (xi < 0) return false;
        if (yi < 0) return true;
        return xv > yv || (xv == yv && xi < yi);
    };
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double ov = __shfl_xor_sync(0xffffffffu, bv, o);
        const long long oi = __shfl_xor_sync(0xffffffffu, bi, o);
        if (better(ov, oi, bv, bi)) { bv = ov; bi = oi; }
    }
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) { sv[wid] = bv; si_[wid] = bi; }
    __syncthreads();
    if (wid == 0) {
        bv = sv[lane]; bi = si_[lane];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double ov = __shfl_xor_sync(0xffffffffu, bv, o);
            const long long oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (better(ov, oi, bv, bi)) { bv = ov; bi = oi; }
        }
        if (lane == 0) out_idx[0] = bi;
    }
}

// PAPER.md:276 "the brute-force Likelihood can ... verify the Heterodyning results": dense log L of each walker
// over the dense bins [i_lo, i_hi) the heterodyne bins cover, template evaluated directly at every bin (no spline,
// no heterodyne), three-term form (Eq. 2-3).  One block per walker; fixed-order reduction.
__global__ void __launch_bounds__(256)
k_het_audit(const double *__restrict__ params, int P, DirectClm cl, StandinInfo si, const double *__restrict__ g4,
            const double *__restrict__ Wd, GridInfo g, const int *__restrict__ estart, int n_b,
            const double *__restrict__ dd, double *__restrict__ logL, double *__restrict__ d_h, double *__restrict__ h_h)
{
    __shared__ double sh[8];
    const size_t w = blockIdx.x;
    const double *rp = params + w * P;
    const int i_lo = estart[0], i_hi = estart[n_b];
    double Mtot, eta, fisco;
    standin_masses(rp[0], rp[1], Mtot, eta, fisco);
    double a_dh = 0.0, a_hh = 0.0;
    for (int i = i_lo + threadIdx.x; i < i_hi; i += blockDim.x) {
        double hAr, hAi, hEr, hEi;
        direct_template_at(rp, cl.c_lm, si, Mtot, eta, fisco, bin_freq(g.k_min, i, g.df), hAr, hAi, hEr, hEi);
        const double4 gg = reinterpret_cast<const double4 *>(g4)[i]; // W conj(d)
        a_dh += (gg.x * hAr - gg.y * hAi) + (gg.z * hEr - gg.w * hEi);
        a_hh = fma(Wd[i], (hAr * hAr + hAi * hAi) + (hEr * hEr + hEi * hEi), a_hh);
    }
    const double t_dh = block_sum_256(a_dh, sh);
    const double t_hh = block_sum_256(a_hh, sh);
    if (threadIdx.x == 0) {
        logL[w] = t_dh - 0.5 * t_hh - 0.5 * dd[1];
        if (d_h) d_h[w] = t_dh;
        if (h_h) h_h[w] = t_hh;
    }
}

// ---------------------------------------------------------------------------------------------------
// H0: heterodyne summary data, one block per bin                   (Eq. 15, 16, 18, 19)
//   A0 = sum W d conj(h0), A1 = sum W d conj(h0)(f - f_b), B0 = sum W |h0|^2, B1 = sum W |h0|^2 (f - f_b)
// raw[b][13]: per channel (A0r, A0i, A1r, A1i, B0, B1), then sum_c W |d|^2 over the bin.
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_het_prepare(const double *__restrict__ g4, const double *__restrict__ Wd, const double *__restrict__ h0, GridInfo g,
              const int *__restrict__ estart, const double *__restrict__ fb, double *__restrict__ raw)
{
    __shared__ double sh[8];
    const int b = blockIdx.x;
    const int i_lo = estart[b], i_hi = estart[b + 1];
    const double f_b = fb[b];
    double acc[13];
#pragma unroll
    for (int q = 0; q < 13; ++q) acc[q] = 0.0;
    for (int i = i_lo + threadIdx.x; i < i_hi; i += blockDim.x) {
        const double4 gg = reinterpret_cast<const double4 *>(g4)[i]; // W conj(d): (W dAr, -W dAi, W dEr, -W dEi)
        const double w = Wd[i];
        const double t = bin_freq(g.k_min, i, g.df) - f_b;
        const double2 ha = reinterpret_cast<const double2 *>(h0)[i];
        const double2 he = reinterpret_cast<const double2 *>(h0)[g.n_f + i];
        // W d conj(h0) = conj( (W conj d) h0 )
        const double par = gg.x * ha.x - gg.y * ha.y, pai = -(gg.x * ha.y + gg.y * ha.x);
        const double per = gg.z * he.x - gg.w * he.y, pei = -(gg.z * he.y + gg.w * he.x);
        const double qa = w * (ha.x * ha.x + ha.y * ha.y), qe = w * (he.x * he.x + he.y * he.y);
        acc[0] += par; acc[1] += pai; acc[2] = fma(par, t, acc[2]); acc[3] = fma(pai, t, acc[3]);
        acc[4] += qa; acc[5] = fma(qa, t, acc[5]);
        acc[6] += per; acc[7] += pei; acc[8] = fma(per, t, acc[8]); acc[9] = fma(pei, t, acc[9]);
        acc[10] += qe; acc[11] = fma(qe, t, acc[11]);
        // W |d|^2 = |W conj d|^2 / W
        if (w > 0.0) acc[12] += (gg.x * gg.x + gg.y * gg.y + gg.z * gg.z + gg.w * gg.w) / w;
    }
#pragma unroll
    for (int q = 0; q < 13; ++q) {
        const double tot = block_sum_256(acc[q], sh);
        if (threadIdx.x == 0) raw[(size_t)b * 13 + q] = tot;
    }
}

// ---------------------------------------------------------------------------------------------------
// H1-H3: heterodyned likelihood.  Packed table (host-built by ll_het_prepare), all in shared memory:
//   edge e : f4[e] = 4 f_e; ih0[e][4] = 1/h0^A (re, im), 1/h0^E (re, im);
//            per mode m: cfp[m][e] = c_lm f_e^(-7/6), f2m[m][e] = 2 f_e/m, fm53[m][e] = (2 f_e/m)^(-5/3)
//   bin b  : A0h[4] = A0/2 (A re, im, E re, im), A1w[4] = A1/(e_{b+1}-e_b), B0q[2] = B0/4, B1w[2] = B1/(e_{b+1}-e_b)
// With s = r_lo + r_hi and dlt = r_hi - r_lo:  r0 = s/2, r1 = dlt/width                         (Eq. 11), so
//   Z[d,h] term = Re[A0 conj r0 + A1 conj r1] = A0h . s + A1w . dlt                              (Eq. 14)
//   Z[h,h] term = B0 |r0|^2 + 2 B1 Re[r0 conj r1] = B0q |s|^2 + B1w (s . dlt)                    (Eq. 17)
// ---------------------------------------------------------------------------------------------------
struct HetTable {
    const double *base; // device copy of the packed table
    int n_e, n_b, n_m;
    int total;          // doubles
    __host__ __device__ int off_f4() const { return 0; }
    __host__ __device__ int off_ih0() const { return n_e; }
    __host__ __device__ int off_cfp() const { return 5 * n_e; }
    __host__ __device__ int off_f2m() const { return 5 * n_e + n_m * n_e; }
    __host__ __device__ int off_fm53() const { return 5 * n_e + 2 * n_m * n_e; }
    __host__ __device__ int off_bins() const { return 5 * n_e + 3 * n_m * n_e; }
};

__device__ __forceinline__ void het_bin_contract(const double *__restrict__ tb, double lAr, double lAi, double lEr,
                                                 double lEi, double hAr, double hAi, double hEr, double hEi,
                                                 double &dh, double &hh)
{
    const double sAr = lAr + hAr, sAi = lAi + hAi, sEr = lEr + hEr, sEi = lEi + hEi;
    const double dAr = hAr - lAr, dAi = hAi - lAi, dEr = hEr - lEr, dEi = hEi - lEi;
    dh = fma(tb[0], sAr, dh); dh = fma(tb[1], sAi, dh); dh = fma(tb[2], sEr, dh); dh = fma(tb[3], sEi, dh);
    dh = fma(tb[4], dAr, dh); dh = fma(tb[5], dAi, dh); dh = fma(tb[6], dEr, dh); dh = fma(tb[7], dEi, dh);
    hh = fma(tb[8], fma(sAr, sAr, sAi * sAi), hh);
    hh = fma(tb[9], fma(sEr, sEr, sEi * sEi), hh);
    hh = fma(tb[10], fma(sAr, dAr, sAi * dAi), hh);
    hh = fma(tb[11], fma(sEr, dEr, sEi * dEi), hh);
}

// Stand-in parameters -> log L.  Block = 32 lanes x (G walker groups x S frequency segments) warps sharing ONE
// copy of the table: warp (g, s) walks segment s of the bins for the 32 walkers of group g.  Lanes of a warp
// are 32 different walkers at the same edge, so every table read is a broadcast.  Blocks stride over passes of
// G groups; the S partial sums of a group meet in shared memory in segment order (deterministic).
//
// Inside a segment the edges go in chunks of E = 4 with the MODE loop outside the edge loop: the transfer factors
// of a mode are read once per chunk (from a lane-major shared copy, so they do not occupy 4 n_m registers for
// the whole kernel), and the four edges of a chunk are four independent phase -> sincos -> T^c h chains in
// flight per thread (with 16 warps per SM the FP64 pipe needs that instruction-level parallelism).  Whether any
// lane needs the taper polynomial is decided once per chunk (warp-uniform), below f_ISCO m_min/2 it is 1.
struct HetEdgeCtx {
    const double *f4, *ih0, *cfp, *f2m, *fm53;
    const double *tfs; // shared: this lane's staged parameter row + 5, i.e. T^c_m (re, im) mode-major, [n_m][4]
    const double *nmq; // shared, [n_m]: -(m/pi)
    int n_e;
    double tc, invD, inv_fisco, K, phi0, kappa, inv_kappa;
};

template <int NM, int E, bool TAPER>
__device__ __forceinline__ void het_eval_edges(const HetEdgeCtx &x, const StandinInfo &si, int e, double (&r)[E][4])
{
    double h[E][4], ftc[E];
#pragma unroll
    for (int k = 0; k < E; ++k) {
        h[k][0] = h[k][1] = h[k][2] = h[k][3] = 0.0;
        ftc[k] = x.f4[e + k] * x.tc;
    }
#pragma unroll 1
    for (int m = 0; m < NM; ++m) {
        const double nmq = x.nmq[m]; // -(m/pi), shared
        const double *tq = x.tfs + m * 4;
        const double t0 = tq[0], t1 = tq[1], t2 = tq[2], t3 = tq[3];
        const int t = m * x.n_e + e;
#pragma unroll
        for (int k = 0; k < E; ++k) {
            // quarter cycles: 4 f t_c + (m/pi) K (2f/m)^(-5/3) - (m/pi)(phi_c + pi/4)
            const double y = fma(x.K, x.fm53[t + k], fma(nmq, x.phi0, ftc[k]));
            double A = x.cfp[t + k] * x.invD;
            if (TAPER) A *= taper_nobranch(x.f2m[t + k] * x.inv_fisco, x.kappa, x.inv_kappa);
            double u, v; // h_m = u - i v
            amp_expi_qc(A, y, u, v);
            h[k][0] = fma(t0, u, h[k][0]); h[k][0] = fma(t1, v, h[k][0]);
            h[k][1] = fma(t1, u, h[k][1]); h[k][1] = fma(-t0, v, h[k][1]);
            h[k][2] = fma(t2, u, h[k][2]); h[k][2] = fma(t3, v, h[k][2]);
            h[k][3] = fma(t3, u, h[k][3]); h[k][3] = fma(-t2, v, h[k][3]);
        }
    }
#pragma unroll
    for (int k = 0; k < E; ++k) { // r = h * (1/h0)
        const double *g = x.ih0 + 4 * (e + k);
        r[k][0] = h[k][0] * g[0] - h[k][1] * g[1];
        r[k][1] = h[k][0] * g[1] + h[k][1] * g[0];
        r[k][2] = h[k][2] * g[2] - h[k][3] * g[3];
        r[k][3] = h[k][2] * g[3] + h[k][3] * g[2];
    }
}

#ifndef LL_HET_E
#define LL_HET_E 4   // edges per chunk (independent chains per thread)
#endif
#ifndef LL_HET_WY
#define LL_HET_WY 16 // warps per block (one block per SM: the table copy is shared by all of them)
#endif
template <int NM>
__global__ void __launch_bounds__(32 * LL_HET_WY)
k_het_standin(HetTable T, StandinInfo si, const double *__restrict__ params, int P, int n_w, int n_groups, int S,
              const double *__restrict__ dd, double *__restrict__ logL, double *__restrict__ d_h,
              double *__restrict__ h_h)
{
    constexpr int E = LL_HET_E;
    extern __shared__ __align__(16) double tab[];
    const int G = blockDim.y / S, seg = threadIdx.y % S, gslot = threadIdx.y / S, lane = threadIdx.x;
    double *red = tab + T.total;                 // [G][S][2][32]
    double *nmq_s = red + (size_t)blockDim.y * 64;   // [8]
    double *tfs_all = nmq_s + 8;                     // [G][32][P]: the parameter rows of the pass
    for (int i = threadIdx.x + threadIdx.y * 32; i < T.total; i += 32 * blockDim.y) tab[i] = T.base[i];
    if (threadIdx.y == 0 && lane < NM) nmq_s[lane] = -((double)si.mode_m[lane] / kPi);
    const int b0 = (int)((long long)seg * T.n_b / S), b1 = (int)((long long)(seg + 1) * T.n_b / S); // balanced to +-1 bin
    HetEdgeCtx x;
    x.f4 = tab + T.off_f4(); x.ih0 = tab + T.off_ih0(); x.cfp = tab + T.off_cfp();
    x.f2m = tab + T.off_f2m(); x.fm53 = tab + T.off_fm53();
    x.nmq = nmq_s;
    x.n_e = T.n_e;
    x.kappa = si.kappa;
    x.inv_kappa = 1.0 / si.kappa;
    const double *bins = tab + T.off_bins();
    const double ddb = dd[1];
    int m_min = si.mode_m[0];
#pragma unroll
    for (int m = 1; m < NM; ++m) m_min = min(m_min, si.mode_m[m]);

    for (int base = blockIdx.x * G; base < n_groups; base += gridDim.x * G) {
        const int grp = base + gslot;
        const int w = grp * 32 + lane;
        const bool valid = grp < n_groups && w < n_w;
        __syncthreads(); // table staged (first pass) / previous pass done with the staged rows and red
        {   // the G x 32 parameter rows of this pass are contiguous in memory: the whole block stages them with
            // coalesced loads (instead of one warp reading 4 n_m strided values per lane while the others wait)
            const long long r0 = (long long)base * 32 * P, r1 = min((long long)(base + G) * 32, (long long)n_w) * P;
            for (long long i = r0 + threadIdx.x + threadIdx.y * 32; i < r1; i += 32 * blockDim.y) tfs_all[i - r0] = params[i];
        }
        __syncthreads();
        const double *row = tfs_all + ((size_t)gslot * 32 + (valid ? lane : 0)) * P; // rows of lanes past n_w: lane 0's
        const WalkerConst c = standin_consts(valid ? row : tfs_all + (size_t)gslot * 32 * P);
        x.tc = c.tc; x.invD = c.invD; x.inv_fisco = c.inv_fisco; x.K = c.K;
        x.phi0 = c.phi + 0.25 * kPi;
        x.tfs = (valid ? row : tfs_all + (size_t)gslot * 32 * P) + 5;
        // x of the lowest-m mode = 2 f/(m_min f_ISCO) = 4 f * x_scale: above 1 somewhere in the warp -> taper needed
        const double x_scale = c.inv_fisco * (0.5 / (double)m_min);
        double dh = 0.0, hh = 0.0;
        if (grp < n_groups && b0 < b1) {
            double pr[1][4];
            if (__any_sync(0xffffffffu, x.f4[b0] * x_scale > 1.0)) het_eval_edges<NM, 1, true>(x, si, b0, pr);
            else het_eval_edges<NM, 1, false>(x, si, b0, pr);
            double pAr = pr[0][0], pAi = pr[0][1], pEr = pr[0][2], pEi = pr[0][3];
            int e = b0 + 1;
            for (; e + E <= b1 + 1; e += E) {
                double r[E][4];
                if (__any_sync(0xffffffffu, x.f4[e + E - 1] * x_scale > 1.0)) het_eval_edges<NM, E, true>(x, si, e, r);
                else het_eval_edges<NM, E, false>(x, si, e, r);
#pragma unroll
                for (int k = 0; k < E; ++k) {
                    het_bin_contract(bins + 12 * (e + k - 1), pAr, pAi, pEr, pEi, r[k][0], r[k][1], r[k][2], r[k][3], dh, hh);
                    pAr = r[k][0]; pAi = r[k][1]; pEr = r[k][2]; pEi = r[k][3];
                }
            }
            for (; e <= b1; ++e) {
                double r[1][4];
                if (__any_sync(0xffffffffu, x.f4[e] * x_scale > 1.0)) het_eval_edges<NM, 1, true>(x, si, e, r);
                else het_eval_edges<NM, 1, false>(x, si, e, r);
                het_bin_contract(bins + 12 * (e - 1), pAr, pAi, pEr, pEi, r[0][0], r[0][1], r[0][2], r[0][3], dh, hh);
                pAr = r[0][0]; pAi = r[0][1]; pEr = r[0][2]; pEi = r[0][3];
            }
        }
        if (S > 1) {
            double *rg = red + (size_t)gslot * S * 64;
            rg[(seg * 2) * 32 + lane] = dh;
            rg[(seg * 2 + 1) * 32 + lane] = hh;
            __syncthreads();
            if (seg == 0) {
                dh = 0.0; hh = 0.0;
                for (int s = 0; s < S; ++s) { dh += rg[(s * 2) * 32 + lane]; hh += rg[(s * 2 + 1) * 32 + lane]; }
            }
        }
        if (seg == 0 && valid) {
            logL[w] = dh - 0.5 * hh - 0.5 * ddb;
            if (d_h) d_h[w] = dh;
            if (h_h) h_h[w] = hh;
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// H1-H3, single mode, regrouped by edge.  With one mode and constant T^c, r^c_e = T^c z_e / h0^c_e with
// z_e = A(f_e) e^{-i Psi(f_e)} common to both channels, and Eq. 14 / Eq. 17 regroup exactly into sums over edges:
//   Z[d,h] = Re sum_c conj(T^c) sum_e conj(z_e) Q^c_e,
//            Q^c_e = conj(1/h0^c_e) (A0_{e-1}/2 + A1_{e-1}/D_{e-1} + A0_e/2 - A1_e/D_e)            (Eq. 11, 14)
//   Z[h,h] = sum_c |T^c|^2 ( sum_e |z_e|^2 P^c_e + sum_b Re[z_b conj(z_{b+1}) X^c_b] ),
//            P^c_e = |1/h0^c_e|^2 (B0_{e-1}/4 + B1_{e-1}/D_{e-1} + B0_e/4 - B1_e/D_e),
//            X^c_b = (B0_b/2) (1/h0^c_b) conj(1/h0^c_{b+1})                                         (Eq. 11, 17)
// (D_b = f_{b+1} - f_b; terms whose bin index falls outside [0, n_b) are absent; 2 Re[r0 conj r1] =
// (|r_hi|^2 - |r_lo|^2)/D.)  Same arithmetic as the bin-by-bin form up to rounding; 48 instead of 73 FP64 slots
// per (walker, bin).  Table: 14 doubles per edge, resident in shared memory, every read a broadcast.
// ---------------------------------------------------------------------------------------------------
constexpr int kHet1Stride = 14; // f4, fm53, cfp, f2m, QAr, QAi, QEr, QEi, PA, PE, XAr, XAi, XEr, XEi

struct Het1Table {
    const double *base;
    int n_e, n_b;
};

#ifndef LL_HET1_WY
#define LL_HET1_WY 16 // warps per block of the single-mode kernel (one block per SM shares the table copy)
#endif
__global__ void __launch_bounds__(32 * LL_HET1_WY)
k_het_standin1(Het1Table T, StandinInfo si, const double *__restrict__ params, int P, int n_w, int n_groups, int S,
               const double *__restrict__ dd, double *__restrict__ logL, double *__restrict__ d_h,
               double *__restrict__ h_h)
{
    extern __shared__ __align__(16) double tab[];
    const int total = T.n_e * kHet1Stride;
    double *red = tab + total; // [G][S][6][32]
    {
        const double2 *src = reinterpret_cast<const double2 *>(T.base);
        double2 *dst = reinterpret_cast<double2 *>(tab);
        for (int i = threadIdx.x + threadIdx.y * 32; i < total / 2; i += 32 * blockDim.y) dst[i] = src[i];
    }
    __syncthreads();
    const int G = blockDim.y / S, seg = threadIdx.y % S, gslot = threadIdx.y / S, lane = threadIdx.x;
    const int per = (T.n_e + S - 1) / S;
    const int e0 = seg * per, e1 = min(e0 + per, T.n_e); // this segment owns edges [e0, e1) and bins [e0, min(e1, n_b))
    const double inv_kappa = 1.0 / si.kappa;
    const double ddb = dd[1];
    const double mh_pi = (double)si.mode_m[0] / kPi;

    for (int base = blockIdx.x * G; base < n_groups; base += gridDim.x * G) {
        const int grp = base + gslot;
        const int w = grp * 32 + lane;
        const bool valid = grp < n_groups && w < n_w;
        const double *row = params + (size_t)(valid ? w : 0) * P;
        const WalkerConst c = standin_consts(row);
        const double Kq = mh_pi * c.K, nphq = -mh_pi * (c.phi + 0.25 * kPi);
        double DAr = 0, DAi = 0, DEr = 0, DEi = 0, HA = 0, HE = 0;
        if (grp < n_groups && e0 < e1) {
            auto edge = [&](const double *t, double &u, double &v, double &amp) {
                const double y = fma(t[0], c.tc, fma(Kq, t[1], nphq));
                amp = t[2] * c.invD * taper(t[3] * c.inv_fisco, si.kappa, inv_kappa);
                amp_expi_qc(amp, y, u, v); // z = u - i v
            };
            const double *t = tab + (size_t)e0 * kHet1Stride;
            double up, vp, ap;
            edge(t, up, vp, ap);
            const int last = min(e1, T.n_b); // one past the last bin whose cross term this segment owns
            auto edge_terms = [&](const double *tt, double u, double v, double a) { // conj(z) Q and |z|^2 P of one edge
                DAr = fma(u, tt[4], DAr); DAr = fma(-v, tt[5], DAr);
                DAi = fma(u, tt[5], DAi); DAi = fma(v, tt[4], DAi);
                DEr = fma(u, tt[6], DEr); DEr = fma(-v, tt[7], DEr);
                DEi = fma(u, tt[7], DEi); DEi = fma(v, tt[6], DEi);
                const double a2 = a * a;
                HA = fma(a2, tt[8], HA);
                HE = fma(a2, tt[9], HE);
            };
            auto cross_terms = [&](const double *tt, double u0, double v0, double u1, double v1) { // z_e conj(z_{e+1}) X
                const double wr = fma(u0, u1, v0 * v1), wi = fma(u0, v1, -(v0 * u1));
                HA = fma(wr, tt[10], HA); HA = fma(-wi, tt[11], HA);
                HE = fma(wr, tt[12], HE); HE = fma(-wi, tt[13], HE);
            };
            int e = e0;
            // chunks of kE bins: the kE next edges are kE independent phase -> sincos chains in flight per thread;
            // the taper polynomial is needed only where some lane is above its f_ISCO (one warp-uniform test per chunk)
            constexpr int kE = 4;
            for (; e + kE <= last; e += kE, t += kE * kHet1Stride) {
                double un[kE], vn[kE], an[kE];
                const bool tapered = __any_sync(0xffffffffu, t[kE * kHet1Stride + 3] * c.inv_fisco > 1.0);
#pragma unroll
                for (int k = 0; k < kE; ++k) {
                    const double *tn = t + (k + 1) * kHet1Stride;
                    const double y = fma(tn[0], c.tc, fma(Kq, tn[1], nphq));
                    double a = tn[2] * c.invD;
                    if (tapered) a *= taper_nobranch(tn[3] * c.inv_fisco, si.kappa, inv_kappa);
                    an[k] = a;
                    amp_expi_qc(a, y, un[k], vn[k]);
                }
#pragma unroll
                for (int k = 0; k < kE; ++k) {
                    const double *tt = t + k * kHet1Stride;
                    const double u0 = k ? un[k - 1] : up, v0 = k ? vn[k - 1] : vp, a0 = k ? an[k - 1] : ap;
                    edge_terms(tt, u0, v0, a0);
                    cross_terms(tt, u0, v0, un[k], vn[k]);
                }
                up = un[kE - 1]; vp = vn[kE - 1]; ap = an[kE - 1];
            }
            for (; e < e1; ++e, t += kHet1Stride) {
                edge_terms(t, up, vp, ap);
                if (e < last) { // bin e = [e, e + 1]: needs z at e + 1 (the next segment's first edge at the boundary)
                    double un, vn, an;
                    edge(t + kHet1Stride, un, vn, an);
                    cross_terms(t, up, vp, un, vn);
                    up = un; vp = vn; ap = an;
                }
            }
        }
        if (S > 1) {
            double *rg = red + (size_t)gslot * S * 192;
            double *q = rg + seg * 192 + lane;
            q[0] = DAr; q[32] = DAi; q[64] = DEr; q[96] = DEi; q[128] = HA; q[160] = HE;
            __syncthreads();
            if (seg == 0) {
                DAr = DAi = DEr = DEi = HA = HE = 0.0;
                for (int s = 0; s < S; ++s) {
                    const double *r = rg + s * 192 + lane;
                    DAr += r[0]; DAi += r[32]; DEr += r[64]; DEi += r[96]; HA += r[128]; HE += r[160];
                }
            }
        }
        if (seg == 0 && valid) {
            const double tar = row[5], tai = row[6], ter = row[7], tei = row[8];
            // Re[conj(T^A) D^A + conj(T^E) D^E],  |T^A|^2 H^A + |T^E|^2 H^E
            const double dh = (tar * DAr + tai * DAi) + (ter * DEr + tei * DEi);
            const double hh = (tar * tar + tai * tai) * HA + (ter * ter + tei * tei) * HE;
            logL[w] = dh - 0.5 * hh - 0.5 * ddb;
            if (d_h) d_h[w] = dh;
            if (h_h) h_h[w] = hh;
        }
        if (S > 1) __syncthreads();
    }
}

// Array entry point: amp_e, phase_e [n_w][n_m][n_e] (radians).  One warp per walker, lanes over edges (the
// arrays are walker-major, so this is the coalesced direction); neighbouring edges meet through a shuffle.
__global__ void __launch_bounds__(256)
k_het_arrays(HetTable T, const double *__restrict__ amp_e, const double *__restrict__ phase_e,
             const double *__restrict__ tf, int n_w, const double *__restrict__ dd, double *__restrict__ logL,
             double *__restrict__ d_h, double *__restrict__ h_h)
{
    extern __shared__ __align__(16) double tab[];
    for (int i = threadIdx.x; i < T.total; i += blockDim.x) tab[i] = T.base[i];
    __syncthreads();
    const double *ih0 = tab + T.off_ih0(), *bins = tab + T.off_bins();
    const int lane = threadIdx.x & 31, wpb = blockDim.x >> 5;
    const double ddb = dd[1];
    for (int w = blockIdx.x * wpb + (threadIdx.x >> 5); w < n_w; w += gridDim.x * wpb) {
        double dh = 0.0, hh = 0.0;
        for (int base = 0; base < T.n_b; base += 31) {
            const int e = base + lane;
            double rAr = 0, rAi = 0, rEr = 0, rEi = 0;
            if (e < T.n_e) {
                double hAr = 0, hAi = 0, hEr = 0, hEi = 0;
                for (int m = 0; m < T.n_m; ++m) {
                    const size_t idx = ((size_t)w * T.n_m + m) * T.n_e + e;
                    const double A = amp_e[idx];
                    double sn, cs;
                    sincos_rad(phase_e[idx], sn, cs);
                    const double u = A * cs, v = A * sn;
                    const double *t4 = tf + ((size_t)w * T.n_m + m) * 4;
                    const double tar = __ldg(t4), tai = __ldg(t4 + 1), ter = __ldg(t4 + 2), tei = __ldg(t4 + 3);
                    hAr = fma(tar, u, hAr); hAr = fma(tai, v, hAr);
                    hAi = fma(tai, u, hAi); hAi = fma(-tar, v, hAi);
                    hEr = fma(ter, u, hEr); hEr = fma(tei, v, hEr);
                    hEi = fma(tei, u, hEi); hEi = fma(-ter, v, hEi);
                }
                const double *g = ih0 + 4 * e;
                rAr = hAr * g[0] - hAi * g[1]; rAi = hAr * g[1] + hAi * g[0];
                rEr = hEr * g[2] - hEi * g[3]; rEi = hEr * g[3] + hEi * g[2];
            }
            const double nAr = __shfl_down_sync(0xffffffffu, rAr, 1), nAi = __shfl_down_sync(0xffffffffu, rAi, 1);
            const double nEr = __shfl_down_sync(0xffffffffu, rEr, 1), nEi = __shfl_down_sync(0xffffffffu, rEi, 1);
            if (lane < 31 && e < T.n_b) het_bin_contract(bins + 12 * e, rAr, rAi, rEr, rEi, nAr, nAi, nEr, nEi, dh, hh);
        }
        dh = warp_sum(dh);
        hh = warp_sum(hh);
        if (lane == 0) {
            logL[w] = dh - 0.5 * hh - 0.5 * ddb;
            if (d_h) d_h[w] = dh;
            if (h_h) h_h[w] = hh;
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// Sampler step around the likelihood (emcee structure, ptemcee tempering, stretch proposal [74];
// readings R25-R28).  The random numbers are inputs.  Proposal arithmetic is written with explicit _rn
// operations (no FMA contraction) so that it is the plain IEEE expression Y = X_j + z (X_k - X_j).
// ---------------------------------------------------------------------------------------------------
// one thread per proposal (t, k): partner j from the other half, z = ((a-1)u+1)^2/a, Y, prior-box test.
// A proposal outside the box is replaced by the walker's own position (so the likelihood kernel sees a valid
// row) and flagged; lnz = (d-1) ln z.
__global__ void __launch_bounds__(128)
k_pt_propose(const double *__restrict__ x, int n_t, int n_w, int P, int half, double a, int n_dim,
             const double *__restrict__ lo, const double *__restrict__ hi, const double *__restrict__ u_z,
             const double *__restrict__ u_partner, double *__restrict__ y, double *__restrict__ lnz,
             int *__restrict__ inside)
{
    const int nh = n_w / 2;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_t * nh) return;
    const int t = i / nh, k = i - t * nh;
    const int k0 = half == 0 ? 0 : nh, j0 = half == 0 ? nh : 0;
    const double tt = __dadd_rn(__dmul_rn(a - 1.0, u_z[i]), 1.0);
    const double z = __ddiv_rn(__dmul_rn(tt, tt), a);
    int j = (int)(u_partner[i] * (double)nh);
    j = min(max(j, 0), nh - 1);
    const double *xk = x + ((size_t)t * n_w + k0 + k) * P;
    const double *xj = x + ((size_t)t * n_w + j0 + j) * P;
    double *yo = y + (size_t)i * P;
    bool in = true;
    for (int q = 0; q < P; ++q) {
        const double v = __dadd_rn(xj[q], __dmul_rn(z, __dadd_rn(xk[q], -xj[q])));
        in = in && (v >= lo[q]) && (v <= hi[q]);
        yo[q] = v;
    }
    if (!in)
        for (int q = 0; q < P; ++q) yo[q] = xk[q];
    inside[i] = in ? 1 : 0;
    lnz[i] = (double)(n_dim - 1) * log(z);
}

// accept when ln u' < (d-1) ln z + beta_t (ln L(Y) - ln L(X_k)), Y inside the box and ln L(Y) finite (R25, R26)
__global__ void __launch_bounds__(128)
k_pt_accept(double *__restrict__ x, double *__restrict__ logL, double *__restrict__ d_h, double *__restrict__ h_h,
            int n_t, int n_w, int P, int half, const double *__restrict__ betas, const double *__restrict__ u_accept,
            const double *__restrict__ y, const double *__restrict__ ly, const double *__restrict__ ydh,
            const double *__restrict__ yhh, const double *__restrict__ lnz, const int *__restrict__ inside,
            int *__restrict__ accepted, unsigned long long *__restrict__ n_acc)
{
    const int nh = n_w / 2;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_t * nh) return;
    const int t = i / nh, k = i - t * nh;
    const size_t wk = (size_t)t * n_w + (half == 0 ? 0 : nh) + k;
    const double l_new = ly[i];
    bool acc = false;
    if (inside[i] && l_new == l_new && fabs(l_new) != INFINITY) {
        const double lnq = __dadd_rn(lnz[i], __dmul_rn(betas[t], __dadd_rn(l_new, -logL[wk])));
        acc = log(u_accept[i]) < lnq;
    }
    if (acc) {
        const double *yo = y + (size_t)i * P;
        double *xo = x + wk * P;
        for (int q = 0; q < P; ++q) xo[q] = yo[q];
        logL[wk] = l_new;
        if (d_h) d_h[wk] = ydh[i];
        if (h_h) h_h[wk] = yhh[i];
    }
    if (accepted) accepted[i] = acc ? 1 : 0;
    if (n_acc && acc) atomicAdd(n_acc + t, 1ull); // integer: order-independent
}

// temperature swaps (R27): one thread per walker column i, rungs swept from the hottest down, sequential in t
__global__ void __launch_bounds__(128)
k_pt_swap(double *__restrict__ x, double *__restrict__ logL, double *__restrict__ d_h, double *__restrict__ h_h,
          int n_t, int n_w, int P, const double *__restrict__ betas, const double *__restrict__ u_swap,
          int *__restrict__ swapped)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_w) return;
    for (int t = n_t - 1; t >= 1; --t) {
        const size_t hi_ = (size_t)t * n_w + i, lo_ = (size_t)(t - 1) * n_w + i;
        const double lh = logL[hi_], lc = logL[lo_];
        const double lnq = __dmul_rn(__dadd_rn(betas[t], -betas[t - 1]), __dadd_rn(lc, -lh));
        const bool sw = log(u_swap[(size_t)(t - 1) * n_w + i]) < lnq;
        if (sw) {
            double *a = x + hi_ * P, *b = x + lo_ * P;
            for (int q = 0; q < P; ++q) { const double v = a[q]; a[q] = b[q]; b[q] = v; }
            logL[hi_] = lc; logL[lo_] = lh;
            if (d_h) { const double v = d_h[hi_]; d_h[hi_] = d_h[lo_]; d_h[lo_] = v; }
            if (h_h) { const double v = h_h[hi_]; h_h[hi_] = h_h[lo_]; h_h[lo_] = v; }
        }
        if (swapped) swapped[(size_t)(t - 1) * n_w + i] = sw ? 1 : 0;
    }
}

// The same sweep with one WARP per walker column for n_t <= 32 and P <= 32 * kSwapRegs... (P <= 64): every row of the
// column is loaded up front (lane q holds coordinate q of each rung; lane t holds ln L, <d|h>, <h|h> and ln u of rung
// t), the cascade then runs on registers and shuffles, and the rows that changed are written back.  Same decisions
// and results as k_pt_swap; the chain of dependent global loads (one per rung) is gone.
__global__ void __launch_bounds__(128)
k_pt_swap_warp(double *__restrict__ x, double *__restrict__ logL, double *__restrict__ d_h, double *__restrict__ h_h,
               int n_t, int n_w, int P, const double *__restrict__ betas, const double *__restrict__ u_swap,
               int *__restrict__ swapped)
{
    const int lane = threadIdx.x & 31;
    const int i = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (i >= n_w) return; // whole warp
    // rung data, one rung per lane
    const bool has = lane < n_t;
    const size_t col = (size_t)(has ? lane : 0) * n_w + i;
    double l = has ? logL[col] : 0.0;
    double dh = (has && d_h) ? d_h[col] : 0.0, hh = (has && h_h) ? h_h[col] : 0.0;
    const double beta = has ? betas[lane] : 0.0;
    const double lnu = (lane >= 1 && has) ? log(u_swap[(size_t)(lane - 1) * n_w + i]) : 0.0; // for the pair (lane, lane-1)
    // coordinates: lane q (and q + 32) of every rung
    double xa[32], xb[32];
#pragma unroll
    for (int t = 0; t < 32; ++t) {
        xa[t] = (t < n_t && lane < P) ? x[((size_t)t * n_w + i) * P + lane] : 0.0;
        xb[t] = (t < n_t && lane + 32 < P) ? x[((size_t)t * n_w + i) * P + lane + 32] : 0.0;
    }
    unsigned changed = 0u;
#pragma unroll
    for (int t = 31; t >= 1; --t) {
        if (t < n_t) { // uniform
            const double lh = __shfl_sync(0xffffffffu, l, t), lc = __shfl_sync(0xffffffffu, l, t - 1);
            const double bh = __shfl_sync(0xffffffffu, beta, t), bc = __shfl_sync(0xffffffffu, beta, t - 1);
            const double lu = __shfl_sync(0xffffffffu, lnu, t);
            const bool sw = lu < __dmul_rn(__dadd_rn(bh, -bc), __dadd_rn(lc, -lh));
            if (sw) {
                const double ta = xa[t]; xa[t] = xa[t - 1]; xa[t - 1] = ta;
                const double tb = xb[t]; xb[t] = xb[t - 1]; xb[t - 1] = tb;
                // rung values live in lanes t and t-1: exchange them
                const double dhh = __shfl_sync(0xffffffffu, dh, t), dhc = __shfl_sync(0xffffffffu, dh, t - 1);
                const double hhh = __shfl_sync(0xffffffffu, hh, t), hhc = __shfl_sync(0xffffffffu, hh, t - 1);
                if (lane == t) { l = lc; dh = dhc; hh = hhc; }
                if (lane == t - 1) { l = lh; dh = dhh; hh = hhh; }
                changed |= (1u << t) | (1u << (t - 1));
            }
            if (swapped && lane == 0) swapped[(size_t)(t - 1) * n_w + i] = sw ? 1 : 0;
        }
    }
#pragma unroll
    for (int t = 0; t < 32; ++t)
        if (t < n_t && ((changed >> t) & 1u)) {
            if (lane < P) x[((size_t)t * n_w + i) * P + lane] = xa[t];
            if (lane + 32 < P) x[((size_t)t * n_w + i) * P + lane + 32] = xb[t];
        }
    if (has && ((changed >> lane) & 1u)) {
        logL[col] = l;
        if (d_h) d_h[col] = dh;
        if (h_h) h_h[col] = hh;
    }
}

// Counter-based uniforms for ll_pt_run_* (reading R31): SplitMix64.  u[kind][index] of iteration `it`:
//   k = mix(seed + G (8 it + kind + 1)),  r = mix(k + G (index + 1)),  u = (r >> 11) 2^-53 in [0, 1)
// kinds 0-2 = u_z, u_partner, u_accept of half 0; 3-5 = of half 1 (n_half = n_t n_w/2 each); 6 = u_swap ((n_t-1) n_w).
__host__ __device__ __forceinline__ unsigned long long splitmix_mix(unsigned long long z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
__global__ void __launch_bounds__(256)
k_pt_uniforms(unsigned long long seed, long long it, int n_half, int n_swap, double *__restrict__ u)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int total = 6 * n_half + n_swap;
    if (i >= total) return;
    const int kind = (i < 6 * n_half) ? i / n_half : 6;
    const int index = i - kind * n_half;
    const unsigned long long G = 0x9E3779B97F4A7C15ull;
    const unsigned long long k = splitmix_mix(seed + G * (unsigned long long)(8 * it + kind + 1));
    const unsigned long long r = splitmix_mix(k + G * (unsigned long long)(index + 1));
    u[i] = (double)(r >> 11) * 0x1.0p-53;
}

// what the stopping tests look at: out[0] = max finite log L, out[1] = its index (lowest on
// ties, -1 if none), out[2] = max extracted SNR <d|h>/sqrt(<h|h>) over entries with <h|h> > 0.  One block.
__global__ void __launch_bounds__(1024)
k_pt_stats(const double *__restrict__ logL, const double *__restrict__ d_h, const double *__restrict__ h_h, long long n,
           double *__restrict__ out)
{
    __shared__ double sv[32], ss[32];
    __shared__ long long si_[32];
    double bv = -INFINITY, bs = -INFINITY;
    long long bi = -1;
    for (long long i = threadIdx.x; i < n; i += blockDim.x) {
        const double v = logL[i];
        if (v == v && fabs(v) != INFINITY && (bi < 0 || v > bv)) { bv = v; bi = i; }
        if (d_h && h_h) {
            const double hh = h_h[i], dh = d_h[i];
            if (hh > 0.0 && dh == dh && fabs(dh) != INFINITY) bs = fmax(bs, dh / sqrt(hh));
        }
    }
    auto better = [](double xv, long long xi, double yv, long long yi) {
        if (xi < 0) return false;
        if (yi < 0) return true;
        return xv > yv || (xv == yv && xi < yi);
    };
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double ov = __shfl_xor_sync(0xffffffffu, bv, o);
        const long long oi = __shfl_xor_sync(0xffffffffu, bi, o);
        if (better(ov, oi, bv, bi)) { bv = ov; bi = oi; }
        bs = fmax(bs, __shfl_xor_sync(0xffffffffu, bs, o));
    }
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) { sv[wid] = bv; si_[wid] = bi; ss[wid] = bs; }
    __syncthreads();
    if (wid == 0) {
        bv = sv[lane]; bi = si_[lane]; bs = ss[lane];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double ov = __shfl_xor_sync(0xffffffffu, bv, o);
            const long long oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (better(ov, oi, bv, bi)) { bv = ov; bi = oi; }
            bs = fmax(bs, __shfl_xor_sync(0xffffffffu, bs, o));
        }
        if (lane == 0) { out[0] = bv; out[1] = (double)bi; out[2] = bs; }
    }
}

// ---------------------------------------------------------------------------------------------------
// ALU roofline denominators: dependent-free FMA chains on every SM (measurement helper)
// ---------------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) k_peak_fma(long long iters, T *__restrict__ sink)
{
    T a[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) a[k] = (T)(threadIdx.x + k) * (T)1e-3;
    const T m = (T)0.999999, c = (T)1e-6;
    for (long long it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int k = 0; k < 8; ++k) a[k] = a[k] * m + c;
    }
    T s = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += a[k];
    if (s == (T)123456.789) sink[0] = s;
}


// operand-pattern variants of the FP64 peak kernel (profiles/: why k_full_fused tops out below 64 DFMA/clk/SM):
//   PAT 0: three distinct, rotating register operands;  PAT 1: one operand from the constant bank
__constant__ double kPeakC[4] = {0.999999, 1e-6, 0.5, 0.25};
template <int PAT>
__global__ void __launch_bounds__(256) k_peak_dfma_pattern(long long iters, double *__restrict__ sink)
{
    double a[8], b[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        a[k] = (double)(threadIdx.x + k) * 1e-3;
        b[k] = 0.9999 + 1e-5 * k + sink[1];
    }
    for (long long it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int k = 0; k < 8; ++k) a[k] = PAT == 0 ? fma(a[k], b[k], a[(k + 3) & 7]) : fma(a[k], b[k], kPeakC[r]);
    }
    double s = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += a[k];
    if (s == 123456.789) sink[0] = s;
}


// issue-mix variants: 32 constant-bank DFMA per iteration plus NI independent integer adds (MIX 0) or binary32
// FMAs (MIX 1) per iteration, in separate dependency chains.  Shows whether instructions for other pipes ride
// along for free while the FP64 pipe is saturated (they do not: profiles/).
template <int MIX, int NI>
__global__ void __launch_bounds__(256) k_peak_dfma_mix(long long iters, double *__restrict__ sink)
{
    double a[8], b[8];
    int q[8];
    float f[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        a[k] = (double)(threadIdx.x + k) * 1e-3;
        b[k] = 0.9999 + 1e-5 * k + sink[1];
        q[k] = threadIdx.x + k;
        f[k] = (float)(threadIdx.x + k) * 1e-3f;
    }
    const int inc = (int)sink[2] + 3;
    const float fm = (float)sink[3] + 0.999f;
    for (long long it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                a[k] = fma(a[k], b[k], kPeakC[r]);
                if ((r * 8 + k) < NI) {
                    if (MIX == 0) asm volatile("add.s32 %0, %0, %1;" : "+r"(q[k]) : "r"(inc));
                    else asm volatile("fma.rn.f32 %0, %0, %1, %1;" : "+f"(f[k]) : "f"(fm));
                }
            }
    }
    double s = 0;
    int t = 0;
    float g = 0.f;
#pragma unroll
    for (int k = 0; k < 8; ++k) { s += a[k]; t += q[k]; g += f[k]; }
    if (s == 123456.789 || t == 123456789 || g == 1234.5f) sink[0] = s;
}

} // namespace ll
