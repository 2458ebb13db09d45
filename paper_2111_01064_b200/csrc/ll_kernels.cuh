// ll_kernels.cuh — the sm_100a kernels of libll_b200 (steps F0-F4, H0-H3 of DESIGN.md §2).
//
// Device layouts ("sorted position" p = index of a walker after the band-top counting sort; n_wp = n_w
// rounded up to the walker-block size):
//   g    [n_f_pad][2 NC]  W^c_i * conj(d^c_i): (re, im) per channel c = A, E(, T); im already negated       (F0)
//   Wc   [NW][n_f_pad]    W^c_i, zero in the padding; NW = 1 (one row shared by all channels) or NC (one per channel)
//   Y    [n_m*2][n_nodes][n_wp]   node values, sys = 2 m + kind (0 amplitude, 1 phase in quarter cycles)
//   C    [n_nodes-1][n_m][8][n_wp] cubic coefficients per interval: (y, b, c, d) amplitude, then phase
//   TF   [n_m][NC][2][n_wp]        transfer factors T^c_m (re, im)
//   part [n_tiles][NQ][n_wp]       per-(frequency tile, walker) partial sums
// Kernels that touch the data tile or the channels are templates on NC (2: A, E; 3: A, E, T — Eq. 3 sums over all
// three) and, where the weights enter, on WS (true: one weight row for every channel, "A=E identical";
// false: one row per channel, "T different").
#pragma once
#include <limits.h>
#include <cooperative_groups.h>
#include "ll_device.cuh"

namespace ll {

constexpr int kMaxModes = 8;
constexpr int kMaxNC = 3;

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

template <int NC>
__global__ void __launch_bounds__(256) k_preweight(const double *__restrict__ d, const double *__restrict__ W, int w_rows,
                                                   int nw_out, long long n_f, long long n_f_pad, double *__restrict__ g,
                                                   double *__restrict__ Wc, double *__restrict__ dd_part)
{
    // d [NC][n_f][2]; W [w_rows][n_f], w_rows = 1 (shared) or NC; g [n_f_pad][2 NC]; Wc [nw_out][n_f_pad] (nw_out = 1
    // needs w_rows = 1; nw_out = NC with w_rows = 1 replicates the row)
    __shared__ double sh[8];
    double acc = 0.0, comp = 0.0; // Neumaier-compensated per-thread sum
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_f; i += (long long)gridDim.x * blockDim.x) {
        double term = 0.0;
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const double w = W[(w_rows > 1 ? (long long)c * n_f : 0) + i];
            const double2 a = reinterpret_cast<const double2 *>(d)[(long long)c * n_f + i];
            reinterpret_cast<double2 *>(g)[i * NC + c] = make_double2(w * a.x, -(w * a.y));
            if (c < nw_out) Wc[(long long)c * n_f_pad + i] = w;
            term = fma(w, a.x * a.x + a.y * a.y, term);
        }
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

// Cost model of the small-batch work partition: one unit per dense bin plus kIntervalCost per spline interval entered
// (an interval change is a dependent load of the coefficients and a re-synchronisation of the recurrence; log-spaced
// nodes put dozens of intervals into the first few hundred bins of the grid).  C(b) = b + K j(b), j(b) = interval of bin b.
constexpr int kIntervalCost = 14;
// (bstart may point to global memory or to a shared-memory copy; nullptr = no shared interval table: C(b) = b)
__device__ __forceinline__ int interval_of_bin_tab(const int *bstart, int n_nodes, int i)
{
    int lo = 0, hi = n_nodes - 2; // largest j in [0, n-2] with bstart[j] <= i
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (bstart[mid] <= i) lo = mid; else hi = mid - 1;
    }
    return lo;
}
__device__ __forceinline__ int cost_of_bin(const int *bstart, int n_nodes, int b)
{
    return bstart ? b + kIntervalCost * interval_of_bin_tab(bstart, n_nodes, b) : b;
}
// smallest bin b with C(b) >= X
__device__ __forceinline__ int first_bin_with_cost(const int *bstart, int n_nodes, int X)
{
    if (!bstart) return X;
    int lo = 0, hi = n_nodes - 2; // largest j with C(bstart[j]) = bstart[j] + K j <= X
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (bstart[mid] + kIntervalCost * mid <= X) lo = mid; else hi = mid - 1;
    }
    const int b = max(bstart[lo], X - kIntervalCost * lo);
    const int end = (lo < n_nodes - 2) ? bstart[lo + 1] : INT_MAX;
    return min(b, end);
}

struct StandinInfo {
    int n_m;
    int m_max;
    int mode_m[kMaxModes];
    double kappa;
    int n_c;      // channels: a parameter row is Mc, q, t_c, phi_c, 1/D, then T^c_m (re, im) mode-major, channel-minor
    int split_tc; // 1: the full-grid node phases are built WITHOUT the linear term 2 pi f t_c, which travels as
                  // t_shift = t_c outside the spline (reading R32)
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
// It also deals the fused kernel's work out by ACTIVE bins (grp_tab, when not null): a group = the 32 walkers of one
// warp (consecutive sorted positions), its bin range [glo, ghi) = union of its walkers' bands, and the n_items blocks
// of the fused kernel are shared among the groups in proportion to ghi - glo, so that every block gets the same
// number of bins of ONE group and all of them start and finish together (no empty tiles, no tail).
// "Bins" are counted in cost units C(b) (above), so that an item of the first, densely noded part of the grid holds
// fewer bins: item t of group g = the bins b of [glo, ghi) with cg + t len <= C(b) < cg + (t + 1) len.
// The kernel is the planner of the whole small-batch call: besides the group table it writes, per item, (group, first
// bin, end bin, interval of the first bin) and, per walker, the first and last item its band touches, so that neither
// the fused kernel's blocks nor k_finalize_small search anything.
constexpr int kGrpStride = 33; // grp_tab: [0..32] first item of group g (entry 32 = total), then glo, ghi, cg, len [32] each,
constexpr int kGrpInts = kGrpStride + 5 * 32; // then the tickets of k_finalize_small [32] (zeroed by the planner)
__host__ __device__ constexpr int grp_off_ticket() { return kGrpStride + 4 * 32; }
// after them: t0[1024], t1[1024] (group items of sorted position p), tb0[1024], tb1[1024] (its own lanes items), then
// item[4][max_items] (group, or -(p + 1) for a lanes item of sorted position p; i0; i1; j0)
__host__ __device__ constexpr int grp_off_t0() { return kGrpInts; }
__host__ __device__ constexpr int grp_off_t1() { return kGrpInts + 1024; }
__host__ __device__ constexpr int grp_off_tb0() { return kGrpInts + 2048; }
__host__ __device__ constexpr int grp_off_tb1() { return kGrpInts + 3072; }
__host__ __device__ constexpr int grp_off_items() { return kGrpInts + 4096; }
// LANES ITEMS (single-mode FP64 kernel).  Inside a group of 32 sorted walkers the band tops differ (by x1.8 in the last
// group of a 160-walker batch), and in group mode a lane whose band has ended rides along idle: measured 1.32x the warp-bins
// a packed batch needs.  So a group's range is split at gsp = the lowest band top of its walkers: [glo, gsp) goes to group
// items as before (every lane active), and the rest goes to lanes items: a SUB-GROUP of kLW neighbouring sorted walkers
// x kLP = 32 / kLW bin phases (k_full_fused's fused_lanes_item): a row of kLP bins per step, idle lanes only where the tops
// inside the sub-group differ.  (kLW = 1, a row of 32 bins of one walker, was measured first and lost: a spline interval is
// then only a few rows long, so the per-lane re-synchronisation is never amortised, and every row pulls 1 KB from L2 for 25
// FP64 instructions — 82 B/clk/SM, more than an SM can draw.  The fewer phases, the longer a lane stays inside one spline
// interval and the fewer bytes a row needs.)  Lanes items are used only where the spline intervals are at
// least kLaneMinInterval bins long.  Cost of a lanes item in the units of the group items: one per row of kLP bins plus
// kLaneIntervalCost per interval.
#ifndef LL_SMALL_LANES
#define LL_SMALL_LANES 1
#endif
#ifndef LL_LANES_WALKERS
#define LL_LANES_WALKERS 16 // 160 walkers on the config-2 grid, fused kernel: no lanes items 0.1454 ms; 4 walkers x 8 phases 0.148
                            // (0.142 with the row cost at 130 %), 8 x 4: 0.147 (0.142), 16 x 2: 0.1291 (row cost 85 %: 0.154,
                            // 110 %: 0.132, 130 %: 0.136); reading the data straight from L2 instead of the TMA ring: 0.142-0.156
#endif
constexpr int kLW = LL_LANES_WALKERS, kLP = 32 / kLW;
#ifndef LL_LANE_INTERVAL_COST
#define LL_LANE_INTERVAL_COST 8
#endif
constexpr int kLaneIntervalCost = LL_LANE_INTERVAL_COST;
#ifndef LL_LANE_ROW_COST
#define LL_LANE_ROW_COST 100
#endif
constexpr int kLaneRowCostPct = LL_LANE_ROW_COST; // cost of a lanes row in percent of a group item's bin
#ifndef LL_LANE_MIN_BINS
#define LL_LANE_MIN_BINS 2048
#endif
constexpr int kLaneMinBins = LL_LANE_MIN_BINS; // a group is split only when its tops differ by more than this
#ifndef LL_LANE_MIN_INTERVAL
#define LL_LANE_MIN_INTERVAL 256
#endif
constexpr int kLaneMinInterval = LL_LANE_MIN_INTERVAL; // and only above the first spline interval at least this long
constexpr int kMinItemCost = 64;
struct BandSortArgs {
    int use_standin;
    const double *params;
    int P;
    const double *band;
    int n_w, n_wp;
    GridInfo g;
    StandinInfo si;
    int *perm, *ilo_s, *ihi_s;
    unsigned long long *pairs;
    int n_items, max_items;
    int *grp_tab;
    const int *bstart_g;
    int n_nodes;
    int lanes; // 1: the fused kernel can take lanes items (single mode, weight moments present)
};
// the body: one block of 1024 threads (k_band_sort_small, or the last block of k_setup_small)
__device__ __forceinline__ void band_sort_small_body(const BandSortArgs &a)
{
    const int use_standin = a.use_standin, P = a.P, n_w = a.n_w, n_wp = a.n_wp, max_items = a.max_items, n_nodes = a.n_nodes;
    const double *__restrict__ params = a.params;
    const double *__restrict__ band = a.band;
    const GridInfo g = a.g;
    const StandinInfo &si = a.si;
    int *__restrict__ perm = a.perm;
    int *__restrict__ ilo_s = a.ilo_s;
    int *__restrict__ ihi_s = a.ihi_s;
    unsigned long long *__restrict__ pairs = a.pairs;
    int n_items = a.n_items;
    int *__restrict__ grp_tab = a.grp_tab;
    const int *__restrict__ bstart_g = a.bstart_g;
    __shared__ int s_hi[1024];
    __shared__ int s_slo[1024], s_shi[1024]; // bands in sorted order
    __shared__ int s_bs[1024];               // the bin -> interval table, when it fits
    __shared__ int s_first[33], s_glo[32], s_ghi[32], s_cg[32], s_len[32];
    __shared__ long long s_U[32];
    __shared__ unsigned long long s_span[32];
    const int w = threadIdx.x;
    const int *bstart = bstart_g;
    if (grp_tab && bstart_g && n_nodes <= 1024) {
        if (w < n_nodes) s_bs[w] = bstart_g[w];
        bstart = s_bs; // visible after the first barrier below
    }
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
        s_slo[rank] = (int)lo;
        s_shi[rank] = (int)hi;
    } else {
        if (w < n_wp) {
            perm[w] = -1;
            ilo_s[w] = 0;
            ihi_s[w] = 0;
        }
        s_slo[w] = 0;
        s_shi[w] = 0;
    }
    if (!grp_tab) return;
    __syncthreads();
    const int n_groups = n_wp >> 5;
    __shared__ long long s_UB;   // cost of all lanes items
    __shared__ int s_lenB, s_totalA, s_nb[1024], s_rb0[1024], s_rb1[1024];
    __shared__ int s_bL; // first bin of the first spline interval of at least kLaneMinInterval bins
    if (w == 0) { s_UB = 0; s_bL = INT_MAX; }
    __syncthreads();
    if (LL_SMALL_LANES && a.lanes && bstart && w < n_nodes - 1 && bstart[w + 1] - bstart[w] >= kLaneMinInterval) atomicMin(&s_bL, bstart[w]);
    for (int j = w + 1024; LL_SMALL_LANES && a.lanes && bstart && j < n_nodes - 1; j += 1024)
        if (bstart[j + 1] - bstart[j] >= kLaneMinInterval) atomicMin(&s_bL, bstart[j]);
    __syncthreads();
    if (w < 32) {
        int glo = INT_MAX, ghi = INT_MIN, gmin = INT_MAX;
        if (w < n_groups)
            for (int k = 0; k < 32; ++k) {
                const int l = s_slo[w * 32 + k], h = s_shi[w * 32 + k];
                if (h > l) { glo = min(glo, l); ghi = max(ghi, h); gmin = min(gmin, h); }
            }
        // group items cover [glo, gsp): up to the lowest band top when the tops differ enough to pay for lanes items
        if (LL_SMALL_LANES && a.lanes && bstart && glo < ghi) {
            const int gsp = max(gmin, min(ghi, s_bL));
            if (ghi - gsp >= kLaneMinBins) ghi = gsp;
        }
        int cg = 0;
        if (glo >= ghi) { glo = 0; ghi = 0; s_U[w] = 0; }
        else {
            cg = cost_of_bin(bstart, n_nodes, glo);
            s_U[w] = (long long)(cost_of_bin(bstart, n_nodes, ghi - 1) - cg + 1);
        }
        grp_tab[kGrpStride + w] = glo;
        grp_tab[kGrpStride + 32 + w] = ghi;
        grp_tab[kGrpStride + 64 + w] = cg;
        grp_tab[grp_off_ticket() + w] = 0;
        s_glo[w] = glo; s_ghi[w] = ghi; s_cg[w] = cg;
    }
    __syncthreads();
    // the rest of a sub-group's bands above its group's items: [rb0, rb1), in lanes items (the sub-group's first thread)
    int rb0 = 0, rb1 = 0, costB = 0;
    if (w < n_wp && (w % kLW) == 0) {
        int l = INT_MAX, h = INT_MIN;
        for (int k = 0; k < kLW; ++k)
            if (s_shi[w + k] > s_slo[w + k]) { l = min(l, s_slo[w + k]); h = max(h, s_shi[w + k]); }
        if (h > l) {
            rb0 = max(l, s_ghi[w >> 5]);
            rb1 = h;
            if (rb1 > rb0)
                costB = (int)(((long long)((rb1 - rb0 + kLP - 1) / kLP) * kLaneRowCostPct) / 100) +
                        kLaneIntervalCost * (interval_of_bin_tab(bstart, n_nodes, rb1 - 1) - interval_of_bin_tab(bstart, n_nodes, rb0) + 1);
            else rb1 = rb0;
        }
    }
    {
        long long cb = costB;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) cb += __shfl_xor_sync(0xffffffffu, cb, o);
        if ((w & 31) == 0 && cb) atomicAdd((unsigned long long *)&s_UB, (unsigned long long)cb); // integers: order-independent
    }
    __syncthreads();
    if (w == 0) {
        long long U = s_UB;
        int n_live = 0;
        for (int k = 0; k < n_groups; ++k) { U += s_U[k]; n_live += s_U[k] > 0; }
        if (U <= 0) U = 1;
        // tiny problems (config 0: 64 walkers x 6.5k bins) take fewer items than the grid has blocks — at least
        // kMinItemCost units each — and the blocks beyond them exit at once
        n_items = (int)max(1LL, min((long long)n_items, max((long long)n_live, U / kMinItemCost)));
        int first = 0;
        for (int k = 0; k < 32; ++k) {
            grp_tab[k] = first;
            s_first[k] = first;
            int n_g = 0;
            if (k < n_groups && s_U[k] > 0) n_g = (int)max(1LL, (long long)n_items * s_U[k] / U);
            const int len = n_g ? (int)((s_U[k] + n_g - 1) / n_g) : 1;
            grp_tab[kGrpStride + 96 + k] = len;
            s_len[k] = len;
            first += n_g;
        }
        s_first[32] = first;
        s_totalA = first;
        s_lenB = (int)max(1LL, (U + n_items - 1) / n_items);
    }
    __syncthreads();
    // lanes items per walker, and their first index (exclusive scan over the sorted positions)
    const int nb = costB ? (costB + s_lenB - 1) / s_lenB : 0;
    s_nb[w] = nb;
    s_rb0[w] = rb0;
    s_rb1[w] = rb1;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) { // inclusive Hillis-Steele scan in shared memory
        const int v = (w >= o) ? s_nb[w - o] : 0;
        __syncthreads();
        s_nb[w] += v;
        __syncthreads();
    }
    const int totalA = s_totalA;
    const int baseB = totalA + s_nb[w] - nb;
    const int total_all = min(totalA + s_nb[1023], max_items);
    if (w == 0) grp_tab[32] = total_all;
    // per item: group, bins [i0, i1), interval of i0
    const int total = min(totalA, max_items);
    int *it = grp_tab + grp_off_items();
    for (int id = w; id < total; id += 1024) {
        int grp = 0;
        while (grp < 31 && s_first[grp + 1] <= id) ++grp;
        const int c0 = s_cg[grp] + (id - s_first[grp]) * s_len[grp];
        const int i0 = min(max(first_bin_with_cost(bstart, n_nodes, c0), s_glo[grp]), s_ghi[grp]);
        const int i1 = min(max(first_bin_with_cost(bstart, n_nodes, c0 + s_len[grp]), s_glo[grp]), s_ghi[grp]);
        it[id] = grp;
        it[max_items + id] = i0;
        it[2 * max_items + id] = i1;
        it[3 * max_items + id] = bstart ? interval_of_bin_tab(bstart, n_nodes, i0) : 0;
    }
    // the lanes items: item k of the sub-group led by sorted position L = an equal share of its [rb0, rb1), in multiples of
    // 32 bins; every thread takes items (the leader of an item by bisection of the scanned counts)
    for (int id = totalA + w; id < total_all; id += 1024) {
        const int rel = id - totalA;
        int lo_ = 0, hi_ = 1023; // smallest L with s_nb[L] > rel
        while (lo_ < hi_) {
            const int mid = (lo_ + hi_) >> 1;
            if (s_nb[mid] > rel) hi_ = mid; else lo_ = mid + 1;
        }
        const int L = lo_, before = L ? s_nb[L - 1] : 0;
        const int nbL = s_nb[L] - before, k = rel - before;
        const int r0 = s_rb0[L], r1 = s_rb1[L];
        const int per = ((r1 - r0 + nbL - 1) / nbL + 31) & ~31;
        const int i0 = min(r0 + k * per, r1), i1 = min(i0 + per, r1);
        it[id] = -(L + 1);
        it[max_items + id] = i0;
        it[2 * max_items + id] = i1;
        it[3 * max_items + id] = interval_of_bin_tab(bstart, n_nodes, i0);
    }
    // per sorted position: first and last group item its band touches, and its own lanes items
    if (w < n_wp) {
        const int grp = w >> 5, l = s_slo[w], h = min(s_shi[w], s_ghi[grp]);
        const int n_g = s_first[grp + 1] - s_first[grp];
        int t0 = 0, t1 = -1;
        if (h > l && n_g > 0) {
            t0 = (cost_of_bin(bstart, n_nodes, l) - s_cg[grp]) / s_len[grp];
            t1 = min((cost_of_bin(bstart, n_nodes, h - 1) - s_cg[grp]) / s_len[grp], n_g - 1);
        }
        grp_tab[grp_off_t0() + w] = s_first[grp] + t0;
        grp_tab[grp_off_t1() + w] = s_first[grp] + t1;
        // its sub-group's lanes items (the scan's values of the sub-group's first thread)
        const int L = w - w % kLW;
        const int incl = s_nb[L], before = L ? s_nb[L - 1] : 0;
        grp_tab[grp_off_tb0() + w] = totalA + before;
        grp_tab[grp_off_tb1() + w] = min(totalA + incl, max_items) - 1;
    }
}

__global__ void __launch_bounds__(1024) k_band_sort_small(BandSortArgs a) { band_sort_small_body(a); }

// exclusive scan of hist[0..n) in place (single block of 1024 threads, n <= 1024*8); starts[0..n] keeps a copy of the
// bucket starts (starts[n] = total), since k_scatter uses hist as its cursors
__global__ void __launch_bounds__(1024) k_scan_hist(int *__restrict__ hist, int n, int *__restrict__ starts)
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
            starts[b + k] = run;
            run += loc[k];
        }
    if (threadIdx.x == 1023) starts[n] = wsum[31];
}

// scatter walkers into their key buckets (order inside a bucket = order of the atomics: NOT reproducible) ...
__global__ void __launch_bounds__(256)
k_scatter(int n_w, const int *__restrict__ key_w, int *__restrict__ offs, int *__restrict__ bucket)
{
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w < n_w) bucket[atomicAdd(&offs[key_w[w]], 1)] = w;
}
// ... and put every bucket into walker order (rank = number of smaller walker indices in the bucket; buckets hold a
// few walkers each), so that the sorted order — hence which walkers share a warp, hence every rounding — is a pure
// function of the inputs and reruns are bit-identical.  One block per bucket; padding positions get perm = -1 and
// an empty band.
constexpr int kSortThreads = 128;
__global__ void __launch_bounds__(kSortThreads)
k_sort_buckets(int n_w, int n_wp, int n_keys, const int *__restrict__ starts, const int *__restrict__ bucket,
               const int *__restrict__ key_w, const int *__restrict__ ilo_w, const int *__restrict__ ihi_w,
               int *__restrict__ perm, int *__restrict__ ilo_s, int *__restrict__ ihi_s)
{
    __shared__ int wtot[kSortThreads / 32];
    const int b = blockIdx.x;
    if (b == n_keys) { // one extra block for the padding
        for (int p = n_w + threadIdx.x; p < n_wp; p += blockDim.x) { perm[p] = -1; ilo_s[p] = 0; ihi_s[p] = 0; }
        return;
    }
    const int s0 = starts[b], s1 = starts[b + 1];
    if (s1 - s0 <= 256) {
        for (int e = s0 + threadIdx.x; e < s1; e += blockDim.x) {
            const int w = bucket[e];
            int rank = 0;
            for (int k = s0; k < s1; ++k) rank += bucket[k] < w;
            perm[s0 + rank] = w;
            ilo_s[s0 + rank] = ilo_w[w];
            ihi_s[s0 + rank] = ihi_w[w];
        }
        return;
    }
    // a big bucket (e.g. every walker with the whole grid as its band): one pass over all walkers in index order,
    // position = start + number of earlier walkers with this key (block-wide running count)
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int base = s0;
    for (int w0 = 0; w0 < n_w; w0 += kSortThreads) {
        const int w = w0 + threadIdx.x;
        const bool mine = w < n_w && key_w[w] == b;
        const unsigned m = __ballot_sync(0xffffffffu, mine);
        if (lane == 0) wtot[wid] = __popc(m);
        __syncthreads();
        int before = __popc(m & ((1u << lane) - 1u)), total = 0;
#pragma unroll
        for (int k = 0; k < kSortThreads / 32; ++k) {
            if (k < wid) before += wtot[k];
            total += wtot[k];
        }
        if (mine) {
            perm[base + before] = w;
            ilo_s[base + before] = ilo_w[w];
            ihi_s[base + before] = ihi_w[w];
        }
        base += total;
        __syncthreads();
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
                y = fma(Kq, nt.fm53[t], -phq);
                if (!si.split_tc) y = fma(nt.f4[j], c.tc, y);
            }
            ya[(size_t)j * n_wp] = a;
            yp[(size_t)j * n_wp] = y;
        }
        if (blockIdx.y == 0) {
            const int nq = 2 * si.n_c;
            for (int q = 0; q < nq; ++q)
                TF[((size_t)m * nq + q) * n_wp + p] = (w >= 0) ? row[5 + m * nq + q] : 0.0;
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
            double y = fma(Kq, nt.fm53[t], -phq);
            if (!si.split_tc) y = fma(nt.f4[j], c.tc, y);
            phase[o] = y * kPio2_1; // quarter cycles -> radians
        }
    }
}

// F1 (array entry point): transpose caller arrays [n_w][n_m][n_nodes] into Y; phase radians -> quarter cycles
__global__ void __launch_bounds__(256)
k_nodes_arrays(const double *__restrict__ amp, const double *__restrict__ phase, const double *__restrict__ tf,
               const int *__restrict__ perm, int n_wp, int n_nodes, int n_m, int n_c, double *__restrict__ Y,
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
        const int nq = 2 * n_c;
        for (int q = 0; q < nq; ++q)
            TF[((size_t)m * nq + q) * n_wp + p0 + tx] = (w >= 0) ? tf[((size_t)w * n_m + m) * nq + q] : 0.0;
    }
}

// F1 (array entry point with a frequency-dependent transfer function, Eq. 8-9): ns = 2 + 2 n_c splines per mode,
// sys = ns m + s with s = 0 amplitude, 1 phase (radians -> quarter cycles), 2 + 2c Re T^c, 3 + 2c Im T^c;
// tf_nodes is [n_w][n_m][n_c][n_nodes][2].  One 32 x 32 transpose tile per block, blockIdx.z = sys.
__global__ void __launch_bounds__(256)
k_nodes_arrays_tf(const double *__restrict__ amp, const double *__restrict__ phase, const double *__restrict__ tf_nodes,
                  const int *__restrict__ perm, int n_wp, int n_nodes, int n_m, int n_c, double *__restrict__ Y)
{
    __shared__ double tt[32][33];
    const int ns = 2 + 2 * n_c;
    const int sys = blockIdx.z, m = sys / ns, s = sys % ns;
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
            else v = tf_nodes[((wm * n_c + ((s - 2) >> 1)) * n_nodes + j) * 2 + ((s - 2) & 1)];
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
#ifndef LL_SPLINE_BLK
#define LL_SPLINE_BLK 24 // rows per register block of both sweeps; config 2: 8 rows 549 us, 16: 518, 24: 447 (254 registers), 32: 477 (spills)
#endif
constexpr int kSplineBlk = LL_SPLINE_BLK;
__global__ void __launch_bounds__(128)
k_spline(const double *__restrict__ Y, double *__restrict__ C, int n_wp, int n_nodes, int n_m, int ns, NodeTables nt)
{
    // ns = splines per mode: 2 (amplitude, phase) or 2 + 2 n_c (+ Re/Im of every T^c: frequency-dependent transfer function)
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
#pragma unroll kSplineBlk
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
// F2 for small batches (Module-1 sized: tens to hundreds of walkers): one block per NWK systems.  With
// few systems the thread-per-system kernel above is a chain of 2 (n-2) dependent steps on a nearly empty GPU.
// Both Thomas sweeps are first-order linear recurrences x_j = alpha_j + beta_j x_{j-1}, i.e. compositions of
// affine maps, which are associative: each thread composes the maps of its ceil(n/T) consecutive rows, a scan
// composes across threads, and each thread then re-runs its rows from the right start value.  Dependent chain:
// 2 ceil(n/T) + scan steps instead of n.  Same factorisation tables; results differ from the sequential sweep
// by rounding only.  Shared memory per warp: node values and dp / M, 2 n doubles.
// ---------------------------------------------------------------------------------------------------
// One block takes NWK (four) neighbouring walkers (sorted positions p0 .. p0 + NWK - 1) of one system: thread =
// (chunk thread ct = tid / 4, walker wl = tid % 4).  With one walker per block every coefficient store and node-value
// load was an isolated 8-byte access (ncu r02: 29 sectors per request, the launch 28 us for 320 systems); with four, a
// row's four walkers are one full 32-byte sector.  STANDIN: the block evaluates its node values from the parameter rows
// itself (the arithmetic of k_nodes_standin; Y is neither written nor read, one launch less) and the amplitude blocks
// write the transfer factors.  Shared memory: ys, ds [n][4] and the exchange slots.
template <int NWK>
__device__ __forceinline__ void affine_scan4_up(double &A, double &B, double *sA, double *sB, int lane, int wid, int nwarp, int wl)
{
#pragma unroll
    for (int o = NWK; o < 32; o <<= 1) {
        const double Ap = __shfl_up_sync(0xffffffffu, A, o), Bp = __shfl_up_sync(0xffffffffu, B, o);
        if (lane >= o) { A = fma(B, Ap, A); B *= Bp; }
    }
    if (lane >= 32 - NWK) { sA[wid * NWK + wl] = A; sB[wid * NWK + wl] = B; }
    __syncthreads();
    double pa = 0.0, pb = 1.0;
    for (int k = 0; k < wid; ++k) { pa = fma(sB[k * NWK + wl], pa, sA[k * NWK + wl]); pb *= sB[k * NWK + wl]; }
    A = fma(B, pa, A);
    B *= pb;
    __syncthreads();
    (void)nwarp;
}
template <int NWK>
__device__ __forceinline__ void affine_scan4_down(double &A, double &B, double *sA, double *sB, int lane, int wid, int nwarp, int wl)
{
#pragma unroll
    for (int o = NWK; o < 32; o <<= 1) {
        const double Ap = __shfl_down_sync(0xffffffffu, A, o), Bp = __shfl_down_sync(0xffffffffu, B, o);
        if (lane + o < 32) { A = fma(B, Ap, A); B *= Bp; }
    }
    if (lane < NWK) { sA[wid * NWK + wl] = A; sB[wid * NWK + wl] = B; }
    __syncthreads();
    double pa = 0.0, pb = 1.0;
    for (int k = nwarp - 1; k > wid; --k) { pa = fma(sB[k * NWK + wl], pa, sA[k * NWK + wl]); pb *= sB[k * NWK + wl]; }
    A = fma(B, pa, A);
    B *= pb;
    __syncthreads();
}

struct Spline4Args {
    const double *Y;
    double *C;
    int n_wp, n_nodes, n_m, ns;
    NodeTables nt;
    const double *params;
    int P;
    const int *perm;
    StandinInfo si;
    double *TF;
};
// wsel[NWK]: the walkers at the block's sorted positions (-1: padding), STANDIN only
template <bool STANDIN, int NWK>
__device__ __forceinline__ void spline_block4_body(const Spline4Args &a, const int *wsel, int block)
{
    const double *__restrict__ Y = a.Y;
    double *__restrict__ C = a.C;
    const int n_wp = a.n_wp, n_nodes = a.n_nodes, n_m = a.n_m, ns = a.ns, P = a.P;
    const NodeTables &nt = a.nt;
    const double *__restrict__ params = a.params;
    const StandinInfo &si = a.si;
    double *__restrict__ TF = a.TF;
    extern __shared__ double ssm[]; // ys[n][4], ds[n][4], xch[T]
    __shared__ double sA[128], sB[128];
    const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31, wid = tid >> 5, nwarp = T >> 5;
    const int wl = tid % NWK, ct = tid / NWK, TT = T / NWK;
    const int nq4 = n_wp / NWK;
    const int sys = block / nq4, p0 = (block - sys * nq4) * NWK;
    const int m = sys / ns, kind = sys % ns;
    const int n = n_nodes;
    const size_t sw = (size_t)n_wp;
    double *ys = ssm, *ds = ys + NWK * n, *xch = ds + NWK * n;
    if (STANDIN) {
        const int w = wsel[wl];
        WalkerConst c = {0, 0, 0, 0, 0};
        const double *row = nullptr;
        if (w >= 0) {
            row = params + (size_t)w * P;
            c = standin_consts(row);
        }
        const double inv_kappa = 1.0 / si.kappa;
        const double mh_pi = (double)si.mode_m[m] / kPi;
        const double phq = mh_pi * (c.phi + 0.25 * kPi), Kq = mh_pi * c.K;
        for (int idx = tid; idx < NWK * n; idx += T) { // idx % NWK = wl
            const int j = idx / NWK;
            const size_t t = (size_t)m * n + j;
            double v = 0.0;
            if (w >= 0) {
                if (kind == 0) v = __ldg(nt.cfp + t) * c.invD * taper(__ldg(nt.f2m + t) * c.inv_fisco, si.kappa, inv_kappa);
                else {
                    v = fma(Kq, __ldg(nt.fm53 + t), -phq);
                    if (!si.split_tc) v = fma(__ldg(nt.f4 + j), c.tc, v);
                }
            }
            ys[idx] = v;
        }
        if (kind == 0) {
            const int nq = 2 * si.n_c;
            if (tid < NWK * nq) { // (q = tid / NWK, walker wl)
                const int q = tid / NWK;
                TF[((size_t)m * nq + q) * sw + p0 + wl] = (w >= 0) ? row[5 + m * nq + q] : 0.0;
            }
        }
    } else {
        for (int idx = tid; idx < NWK * n; idx += T) ys[idx] = __ldg(Y + ((size_t)sys * n + idx / NWK) * sw + p0 + wl);
    }
    __syncthreads();
    const int L = (n + TT - 1) / TT;
    const int j0 = min(ct * L, n), j1 = min(j0 + L, n);
    auto yv = [&](int j) { return ys[NWK * j + wl]; };
    auto rhs = [&](int j) { return (yv(j + 1) - yv(j)) * __ldg(nt.invh + j) - (yv(j) - yv(j - 1)) * __ldg(nt.invh + j - 1); };
    // ---- forward sweep: dp_j = (r_j - a_j dp_{j-1}) / den_j for j = 1..n-2, dp_0 = 0
    double A = 0.0, B = 1.0;
    for (int j = j0; j < j1; ++j)
        if (j >= 1 && j <= n - 2) {
            const double ti = __ldg(nt.tinv + j), be = -__ldg(nt.ta + j) * ti;
            A = fma(be, A, rhs(j) * ti);
            B *= be;
        }
    affine_scan4_up<NWK>(A, B, sA, sB, lane, wid, nwarp, wl);
    xch[tid] = A;
    __syncthreads();
    double start = ct ? xch[tid - NWK] : 0.0;
    for (int j = j0; j < j1; ++j) {
        if (j >= 1 && j <= n - 2) start = (rhs(j) - __ldg(nt.ta + j) * start) * __ldg(nt.tinv + j);
        ds[NWK * j + wl] = (j >= 1 && j <= n - 2) ? start : 0.0;
    }
    __syncthreads();
    // ---- backward sweep: M_j = dp_j - c'_j M_{j+1} for j = n-2..1, M_0 = M_{n-1} = 0
    A = 0.0; B = 1.0;
    for (int j = j1 - 1; j >= j0; --j) {
        if (j >= 1 && j <= n - 2) {
            const double be = -__ldg(nt.tcp + j);
            A = fma(be, A, ds[NWK * j + wl]);
            B *= be;
        } else { A = 0.0; B = 0.0; }
    }
    affine_scan4_down<NWK>(A, B, sA, sB, lane, wid, nwarp, wl);
    xch[tid] = A;
    __syncthreads();
    double Mn = (ct + 1 < TT) ? xch[tid + NWK] : 0.0;
    for (int j = j1 - 1; j >= j0; --j) {
        Mn = (j >= 1 && j <= n - 2) ? fma(-__ldg(nt.tcp + j), Mn, ds[NWK * j + wl]) : 0.0;
        ds[NWK * j + wl] = Mn;
    }
    __syncthreads();
    if (nt.bc) { // not-a-knot end values from their neighbours
        if (ct == 0) {
            ds[wl] = (1.0 + nt.rho0) * ds[NWK + wl] - nt.rho0 * ds[2 * NWK + wl];
            ds[NWK * (n - 1) + wl] = (1.0 + nt.rhon) * ds[NWK * (n - 2) + wl] - nt.rhon * ds[NWK * (n - 3) + wl];
        }
        __syncthreads();
    }
    // ---- coefficients of interval j (same formulas as k_spline): four walkers of a row = one 32-byte sector per store
    double *c = C + ((size_t)m * ns * 4 + kind * 4) * sw + p0 + wl;
    const size_t cj = (size_t)n_m * ns * 4 * sw;
    for (int idx = tid; idx < NWK * (n - 1); idx += T) {
        const int j = idx / NWK;
        const double y0 = ys[idx], y1 = ys[idx + NWK], Mj = ds[idx], Mn1 = ds[idx + NWK];
        const double h = __ldg(nt.hj + j), ih = __ldg(nt.invh + j);
        double *cc = c + (size_t)j * cj;
        cc[0] = y0;
        cc[sw] = (y1 - y0) * ih - h * (2.0 * Mj + Mn1) * kSixth;
        cc[2 * sw] = 0.5 * Mj;
        cc[3 * sw] = (Mn1 - Mj) * ih * kSixth;
    }
}

template <bool STANDIN, int NWK>
__global__ void __launch_bounds__(1024) k_spline_block4(Spline4Args a)
{
    __shared__ int s_wsel[NWK];
    if (STANDIN) {
        if (threadIdx.x < NWK) s_wsel[threadIdx.x] = a.perm[(blockIdx.x % (a.n_wp / NWK)) * NWK + threadIdx.x];
        __syncthreads();
    }
    spline_block4_body<STANDIN, NWK>(a, s_wsel, blockIdx.x);
}

// The whole set-up of a small stand-in batch in ONE launch of 1024-thread blocks: the last block is the planner
// (band_sort_small_body: bands, sort, cost plan of the fused kernel), every other block is a spline block that does
// not wait for the planner's sort — it ranks the walkers itself (every thread one band top, the same band_bins and
// the same (top, index) order as the planner, so the two agree exactly) and keeps the NWK walkers whose ranks are its
// sorted positions.  Three launches per call (set-up, fused, F4) instead of four.
template <int NWK>
__global__ void __launch_bounds__(1024) k_setup_small(Spline4Args a, BandSortArgs b)
{
    if (blockIdx.x == gridDim.x - 1) {
        band_sort_small_body(b);
        return;
    }
    __shared__ int s_top[1024];
    __shared__ int s_wsel[NWK];
    const int w = threadIdx.x;
    long long lo = 0, hi = 0;
    if (w < b.n_w) band_bins(b.use_standin, b.params, b.P, b.band, w, b.g, b.si, lo, hi);
    s_top[w] = (w < b.n_w) ? (int)hi : INT_MAX;
    if (w < NWK) s_wsel[w] = -1;
    __syncthreads();
    const int p0 = (blockIdx.x % (a.n_wp / NWK)) * NWK;
    if (w < b.n_w) {
        const int mine = (int)hi;
        int rank = 0;
        for (int k = 0; k < b.n_w; ++k) {
            const int other = s_top[k];
            rank += (other < mine) || (other == mine && k < w);
        }
        if (rank >= p0 && rank < p0 + NWK) s_wsel[rank - p0] = w;
    }
    __syncthreads();
    spline_block4_body<true, NWK>(a, s_wsel, blockIdx.x);
}

// ---------------------------------------------------------------------------------------------------
// F3: fused spline evaluation / channel response / inner products           (Eq. 3, 7, 9)
// One thread = one walker; a warp = 32 walkers walking the SAME dense bins, so the data tile (g, W) is a
// shared-memory broadcast and no cross-thread reduction exists.  Tiles of g/W arrive by 1-D bulk TMA into
// a two-stage ring guarded by mbarriers.  The dense template is never written anywhere.
// Single-mode specialisation: T^c is constant per walker, so the kernel accumulates the complex sums
// S^c = sum_i g^c_i A e^{-i Psi} and H = sum_i W_i A^2; k_finalize applies T^c.
// ---------------------------------------------------------------------------------------------------
// Prefix moments of the (shared) weight row inside each spline interval, for the single-mode kernel's <h|h>:
// inside an interval A(t) is a cubic in t = f - x_j, so sum_k W_k A(t_k)^2 over any stretch of its bins is
// sum_{p=0..6} q_p M_p with q = the coefficients of A^2 and M_p = sum_k W_k t_k^p — walker-independent sums.
//   wmom[p][i] = sum over the bins k of bin i's interval, k <= i, of W_k t_k^p          (inclusive prefix)
// so M_p of a stretch [b0, b1) of one interval is wmom[p][b1 - 1] - wmom[p][b0 - 1] (the second term absent when b0 is
// the interval's first bin).  One block per interval; t exactly as the fused kernel forms it.  Rebuilt when the node
// set or the data change.  A prefix over an interval of n bins carries ~sqrt(n) ulp, the difference of two of them the
// same absolutely: 1e-15 relative to a stretch a fortieth of its interval — the 1e-12 the log L = 0 test needs is far.
__global__ void __launch_bounds__(256)
k_w_moments(const double *__restrict__ Wc, const int *__restrict__ bstart, const double *__restrict__ xj, int n_nodes,
            long long k_min, double df, long long n_f_pad, double *__restrict__ wmom)
{
    __shared__ double wtot[8][7];
    const int j = blockIdx.x;
    Wc += (size_t)blockIdx.y * n_f_pad;          // weight row blockIdx.y
    wmom += (size_t)blockIdx.y * 7 * n_f_pad;    // and its seven prefix rows
    const int i0 = bstart[j], i1 = bstart[j + 1];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const double nx = -xj[j];
    double carry[7];
#pragma unroll
    for (int p = 0; p < 7; ++p) carry[p] = 0.0;
    for (int base = i0; base < i1; base += 256) {
        const int i = base + threadIdx.x;
        double v[7];
        {
            const double t = fma((double)(k_min + i), df, nx);
            double w = (i < i1) ? Wc[i] : 0.0;
#pragma unroll
            for (int p = 0; p < 7; ++p) { v[p] = w; w *= t; }
        }
#pragma unroll
        for (int p = 0; p < 7; ++p) { // inclusive scan inside the warp
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const double u = __shfl_up_sync(0xffffffffu, v[p], o);
                if (lane >= o) v[p] += u;
            }
        }
        if (lane == 31) {
#pragma unroll
            for (int p = 0; p < 7; ++p) wtot[wid][p] = v[p];
        }
        __syncthreads();
#pragma unroll
        for (int p = 0; p < 7; ++p) {
            double pre = carry[p], tot = carry[p];
            for (int k = 0; k < 8; ++k) {
                if (k < wid) pre += wtot[k][p];
                tot += wtot[k][p];
            }
            if (i < i1) wmom[(size_t)p * n_f_pad + i] = pre + v[p];
            carry[p] = tot;
        }
        __syncthreads();
    }
}

struct FusedArgs {
    const double *g;       // [n_f_pad][2 NC]
    const double *Wc;      // [NW][n_f_pad]
    const double *C;
    const double *TF;
    const double *xj;
    const int *bstart;
    const int *ilo;
    const int *ihi;
    const int *perm;       // sorted position -> walker index (t_shift is in the caller's order), -1 in the padding
    const double *t_shift; // t_shift of walker w at t_shift[w * ts_stride] (seconds), or nullptr:
    int ts_stride;         // Psi_m(f) = spline_m(f) + 2 pi f t_shift (reading R32); the stand-in passes params + 2, P
    double *part;
    long long k_min;
    long long n_f_pad;     // row stride of Wc
    double df;
    const int *tile_start; // [n_tiles + 1]: frequency tile t covers dense bins [tile_start[t], tile_start[t+1])
    const int *grp_tab;    // small batches (k_full_fused<.., SMALL = 1>): work dealt out by active bins, see k_band_sort_small
    const double *wmom;    // [NW][7][n_f_pad] prefix moments of every weight row inside each spline interval (k_w_moments), or null
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

// One stage of the data ring in shared memory: the g tile [CH][2 NC], then NW weight rows [CH] — (2 NC + NW) doubles
// per bin, 1 + NW bulk copies per stage, all completing on the stage's mbarrier.
template <int NC, bool WS>
struct Tile {
    static constexpr int NW = WS ? 1 : NC;
    static constexpr int DPB = 2 * NC + NW; // doubles per bin
    __device__ static __forceinline__ void issue(const FusedArgs &a, double *dst, int c, int CH, uint64_t *bar)
    {
        mbar_expect_tx(bar, (uint32_t)CH * 8u * DPB);
        tma_load_1d(dst, a.g + (size_t)c * CH * 2 * NC, (uint32_t)CH * 16u * NC, bar);
#pragma unroll
        for (int r = 0; r < NW; ++r)
            tma_load_1d(dst + (size_t)CH * (2 * NC + r), a.Wc + (size_t)r * a.n_f_pad + (size_t)c * CH, (uint32_t)CH * 8u, bar);
    }
};

// LL_POISON_STAGES (a test build; compute-sanitizer is closed on this pool): when a block has finished with a stage of
// the ring, it overwrites the stage with NaNs before the barrier that frees it for the next bulk copy.  A thread that
// read a stage before its copy had landed — a wrong mbarrier phase, a missing wait — would then see NaNs instead of the
// previous tile's plausible numbers, and every parity test would fail.  The generic-proxy stores are ordered before
// the async-proxy copy that refills the stage by fence.proxy.async.
__device__ __forceinline__ void poison_stage(const double *stage, int n_doubles)
{
#ifdef LL_POISON_STAGES
    __syncthreads(); // the other warps of the block may still be reading the stage
    double *w = const_cast<double *>(stage);
    for (int i = threadIdx.x; i < n_doubles; i += blockDim.x) w[i] = __longlong_as_double(0x7ff8000000000000LL);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
#else
    (void)stage; (void)n_doubles;
#endif
}

// g of bin ii from a tile pointer that has been moved back by the tile's first bin (sgc = tile - cb * 2 NC)
template <int NC>
__device__ __forceinline__ void load_g(const double *__restrict__ sgc, int ii, double (&g)[2 * NC])
{
    if (NC == 2) {
        const double4 v = reinterpret_cast<const double4 *>(sgc)[ii];
        g[0] = v.x; g[1] = v.y; g[2] = v.z; g[3] = v.w;
    } else {
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const double2 v = reinterpret_cast<const double2 *>(sgc)[ii * NC + c];
            g[2 * c] = v.x; g[2 * c + 1] = v.y;
        }
    }
}

// accumulators of the single-mode kernel: S^c = sum_i g^c_i A e^{-i Psi} (complex, per channel) and
// H = sum_i W_i A^2 (one for a shared weight row, one per channel otherwise); k_finalize applies T^c.
template <int NC, bool WS>
struct Acc1 {
    static constexpr int NW = WS ? 1 : NC;
    double S[2 * NC];
    double H[NW];
    __device__ __forceinline__ void zero()
    {
#pragma unroll
        for (int q = 0; q < 2 * NC; ++q) S[q] = 0.0;
#pragma unroll
        for (int q = 0; q < NW; ++q) H[q] = 0.0;
    }
    // h = u - i v = A e^{-i Psi} at bin ii; WITH_H = false: the stretch's sum of W A^2 comes from the weight moments
    template <bool WITH_H = true>
    __device__ __forceinline__ void add(const double *__restrict__ sgc, const double *__restrict__ sWc, int CH, int ii,
                                        double u, double v, double A)
    {
        double g[2 * NC];
        load_g<NC>(sgc, ii, g);
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            S[2 * c] = fma(g[2 * c], u, S[2 * c]); S[2 * c] = fma(g[2 * c + 1], v, S[2 * c]);
            S[2 * c + 1] = fma(g[2 * c + 1], u, S[2 * c + 1]); S[2 * c + 1] = fma(-g[2 * c], v, S[2 * c + 1]);
        }
        if (!WITH_H) return;
        if (WS) {
            H[0] = fma(sWc[ii] * A, A, H[0]);
        } else {
            const double A2 = A * A;
#pragma unroll
            for (int c = 0; c < NC; ++c) H[c] = fma(sWc[c * CH + ii], A2, H[c]);
        }
    }
};

// <d|h> and <h|h> contributions of one bin given the channel responses h^c = (hr, hi) (kernels that apply T^c per bin)
template <int NC, bool WS>
__device__ __forceinline__ void accumulate_bin(const double *__restrict__ sgc, const double *__restrict__ sWc, int CH, int ii,
                                               const double (&h)[2 * NC], double &s_dh, double &s_hh)
{
    double g[2 * NC];
    load_g<NC>(sgc, ii, g);
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        s_dh = fma(g[2 * c], h[2 * c], s_dh);
        s_dh = fma(-g[2 * c + 1], h[2 * c + 1], s_dh);
    }
    if (WS) {
        double q = fma(h[0], h[0], h[1] * h[1]);
#pragma unroll
        for (int c = 1; c < NC; ++c) q += fma(h[2 * c], h[2 * c], h[2 * c + 1] * h[2 * c + 1]);
        s_hh = fma(sWc[ii], q, s_hh);
    } else {
#pragma unroll
        for (int c = 0; c < NC; ++c)
            s_hh = fma(sWc[c * CH + ii], fma(h[2 * c], h[2 * c], h[2 * c + 1] * h[2 * c + 1]), s_hh);
    }
}

// h^c += T^c (u - i v) for every channel; T^c = (tf[2c], tf[2c+1])
template <int NC>
__device__ __forceinline__ void apply_tf(const double (&tf)[2 * NC], double u, double v, double (&h)[2 * NC])
{
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        h[2 * c] = fma(tf[2 * c], u, h[2 * c]); h[2 * c] = fma(tf[2 * c + 1], v, h[2 * c]);
        h[2 * c + 1] = fma(tf[2 * c + 1], u, h[2 * c + 1]); h[2 * c + 1] = fma(-tf[2 * c], v, h[2 * c + 1]);
    }
}

// Linear phase term outside the spline (reading R32): Psi(f) = spline(f) + 2 pi f t_shift, i.e. 4 f t_shift quarter
// cycles.  It is folded into the phase cubic of the current interval: with f = x_j + t,
//   c0 += 4 t_shift x_j (taken modulo one cycle: e^{-i Psi} does not see whole cycles),   c1 += 4 t_shift,
// so neither route pays anything per bin.  The product is formed exactly (hi + lo by FMA) and the whole cycles are
// removed from hi before the sum, so the large linear phase (1e7 quarter cycles at the top of a one-year band) never
// costs the low bits of the small splined one.
__device__ __forceinline__ double qc_linear_mod_cycle(double x, double ts4 /* 4 t_shift */)
{
    const double hi = ts4 * x, lo = fma(ts4, x, -hi);
    const double n4 = 4.0 * rint(0.25 * hi); // whole cycles, in quarter cycles; hi - n4 is exact
    return (hi - n4) + lo;
}

#ifndef LL_FUSED_UNROLL
#define LL_FUSED_UNROLL 3 // bins in flight per thread in the hot loop (tuned on B200, profiles/)
#endif
#ifndef LL_FUSED_MINB
#define LL_FUSED_MINB 6 // resident 128-thread blocks per SM the register budget of the single-mode large-batch kernel is held
                        // to: 80 registers (the multi-mode and small-batch instantiations keep 4: 128).  Measured at
                        // config 2 (round 2, 256-bin stages): 4 blocks (118 registers) 9.37 ms, 5 (96) 9.57, 6 (80, ~50 bytes
                        // of spills outside the bin loop) 9.17, 7 (72) 9.44; with 512-bin stages (five blocks fit the shared
                        // memory) and the recurrence loop unrolled four times: 8.99 ms
#endif
#ifndef LL_FUSED_MINB_SMALL
#define LL_FUSED_MINB_SMALL 4 // register budget of the small-batch instantiation (one-warp blocks), as blocks of 128 threads
#endif
#ifndef LL_FUSED_MINB_PC
#define LL_FUSED_MINB_PC 4 // the same for the layouts with per-channel weight rows: three channels at config-2 size 11.08 ms at 3 blocks (160 registers), 10.96 at 4 (128), 11.57 at 5 (96)
#endif
constexpr int kFusedUnroll = LL_FUSED_UNROLL;
// bins [b0, b1) of one spline interval for the single-mode kernel: t, the two cubics, A e^{-i Psi}, the complex MACs
// with g^c and W A^2.  MASK = per-lane band test (only at the ragged ends of a warp's band).
template <bool MASK, int NC, bool WS>
__device__ __forceinline__ void fused_bins_nm1(int b0, int b1, int tlo, int thi, int kbase, double df, double nxj,
                                               double cA0, double cA1, double cA2, double cA3, double cP0, double cP1,
                                               double cP2, double cP3, const double *__restrict__ sgc,
                                               const double *__restrict__ sWc, int CH, Acc1<NC, WS> &acc)
{
#pragma unroll kFusedUnroll
    for (int ii = b0; ii < b1; ++ii) {
        const double t = fma((double)(kbase + ii), df, nxj);
        double A = fma(fma(fma(cA3, t, cA2), t, cA1), t, cA0);
        const double y = fma(fma(fma(cP3, t, cP2), t, cP1), t, cP0);
        if (MASK) A = ((ii >= tlo) && (ii < thi)) ? A : 0.0;
        double u, v; // h = u - i v
        amp_expi_qc(A, y, u, v);
        acc.add(sgc, sWc, CH, ii, u, v, A);
    }
}

// The same bins by recurrence (SURVEY.md "hard parts"; unmasked bins of one spline interval only).  On the uniform
// grid the phase cubic has constant third differences, so e^{-i Psi_k} advances by three complex rotations per bin,
//   z_{k+1} = z_k w_k,  w_{k+1} = w_k v_k,  v_{k+1} = v_k u,   w = e^{i D1 Psi}, v = e^{i D2 Psi}, u = e^{i D3 Psi},
// and the amplitude cubic by its forward differences; every kRotSync bins everything is re-evaluated from the cubic
// coefficients, which bounds the accumulated rounding: with D1 Psi <= a few quarter cycles known to 1 ulp, the phase
// drifts by < kRotSync^2/2 ulp ~ 1e-12 quarter cycles between re-syncs, far below the rounding of Psi itself (1e-9 at
// 1e7 quarter cycles) — PROVIDED the rotations w, v, u themselves carry no systematic error (LL_ROT_ACC, ll_device.cuh).  Per bin: 12 (rotations) + 3 (amplitude) + 2 (A z) + 4 NC
// (MACs) + 2 (W A^2; 1 + NC with per-channel weights) = 27 FP64 instructions for two channels and a shared weight row
// (33 for three channels with their own rows), no sincos, no quadrant fix-up, no bin-number conversion, instead of
// 34 + 18 others.
#ifndef LL_FUSED_ROT
#define LL_FUSED_ROT 1
#endif
#ifndef LL_H_MOMENTS
#define LL_H_MOMENTS 1 // <h|h> of an unmasked recurrence stretch from prefix moments of the weights (k_w_moments)
#endif
#ifndef LL_ROT_SYNC
#define LL_ROT_SYNC 128 // bins between re-synchronisations.  Measured at config 2 (max |<d|h> - oracle| over 25 sampled
                        // walkers at <d|h> up to 2.5e5; kernel time).  Round 1, rotations from the degree-5 polynomials:
                        // 32: 8e-8, 10.7 ms; 64: 3e-7; 128: 2e-6; 256: 1.3e-5 — the error grew like the length squared
                        // because the polynomial's phase error in w is amplified k-fold in z and has the same sign over
                        // thousands of blocks.  Round 2, rotations from the degree-7 polynomials (LL_ROT_ACC): 32: 9e-8,
                        // 10.9 ms; 64: 1.1e-7, 10.35; 128: 1.3e-7, 10.09 (chosen; noiseless log L at the truth -1.6e-8);
                        // 256: 1.2e-7, 9.96 (noiseless -8.7e-8).  The exact route: 7e-8, 13.0 ms.
#endif
#ifndef LL_ROT_UNROLL
#define LL_ROT_UNROLL 4 // bins per trip of the unmasked recurrence loop in large batches (2 for the masked ends and small batches)
#endif
#ifndef LL_ROT_ACC
#define LL_ROT_ACC 1 // the rotations of a re-synchronisation from the degree-7 polynomials (ll_device.cuh)
#endif
#if LL_ROT_ACC
#define LL_ROT_SINCOS sincos_qc_acc
#else
#define LL_ROT_SINCOS sincos_qc
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
// MASK: lanes outside their own band [tlo, thi) ride along with amplitude 0 (the ragged end of a warp's band: a
// few bins in a large sorted batch, but a third of all bins when a whole batch is only a handful of warps).
template <bool MASK, int NC, bool WS, bool WITH_H = true, int UNR = 2>
__device__ __forceinline__ void fused_bins_rot(int b0, int b1, int tlo, int thi, int kbase, double df, double nxj, double cA0,
                                               double cA1, double cA2, double cA3, double cP0, double cP1, double cP2,
                                               double cP3, const double *__restrict__ sgc, const double *__restrict__ sWc,
                                               int CH, Acc1<NC, WS> &acc)
{
    const double df2 = df * df, df3 = df2 * df;
    const double d3A = 6.0 * cA3 * df3;
    double su, cu;
    LL_ROT_SINCOS(6.0 * cP3 * df3, su, cu);
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
        LL_ROT_SINCOS(fma(fma(fma(cP3, t, cP2), t, cP1), t, cP0), sz, cz);
        LL_ROT_SINCOS(df * fma(cP3, q3, fma(cP2, tt, cP1)), sw, cw);
        LL_ROT_SINCOS(df2 * fma(6.0 * cP3, t1, 2.0 * cP2), sv, cv);
        unit_modulus(cz, sz);
        unit_modulus(cw, sw);
        unit_modulus(cv, sv);
#pragma unroll UNR
        for (int ii = k0; ii < k1; ++ii) {
            const double Am = (!MASK || ((ii >= tlo) && (ii < thi))) ? A : 0.0;
            const double u = Am * cz, v = Am * sz; // h = u - i v
            acc.template add<WITH_H>(sgc, sWc, CH, ii, u, v, Am);
            const double nzc = fma(cz, cw, -(sz * sw)), nzs = fma(sz, cw, cz * sw);
            const double nwc = fma(cw, cv, -(sw * sv)), nws = fma(sw, cv, cw * sv);
            const double nvc = fma(cv, cu, -(sv * su)), nvs = fma(sv, cu, cv * su);
            cz = nzc; sz = nzs; cw = nwc; sw = nws; cv = nvc; sv = nvs;
            A += d1A; d1A += d2A; d2A += d3A;
        }
    }
}

// A LANES ITEM of the small-batch kernel (planner: band_sort_small_body's lanes items): bins [i0, i1) of the kLW walkers at
// sorted positions p0 .. p0 + kLW - 1.  Lane = (walker wl = lane % kLW, bin phase ph = lane / kLW): row r holds the bins
// kLP r .. kLP r + kLP - 1, and a lane always takes the bins = ph (mod kLP) of its walker — a uniform sequence of stride
// kLP df, so inside one spline interval it advances e^{-i Psi} and A by the recurrence of fused_bins_rot with df -> kLP df
// (its own z, w, v, u and amplitude differences), re-synchronised from the walker's cubic coefficients every kLaneSync
// rows and at every interval; outside its walker's band, or the stretch, a lane carries amplitude 0.  <h|h> of a walker's
// stretch comes from the weight moments (one evaluation per stretch, added by the walker's phase-0 lane).  The data are
// read straight from L2/L1 (a row is kLP x 2 NC doubles, each broadcast to kLW lanes), not through the TMA ring.  At the
// end the phases of a walker are added by a butterfly (a fixed order) and its phase-0 lane writes the walker's slot of
// the item's record.
constexpr int kLaneSync = 128;
template <int NC, bool WS>
__device__ __forceinline__ void fused_lanes_item(const FusedArgs &a, int pw, int lo, int hi, int wlo, int whi, int j, int item,
                                                 double *sm, uint64_t *bar)
{
    // pw: this lane's walker, [lo, hi): its bins in the item (empty: lo >= hi), [wlo, whi): the union over the warp
    using TL = Tile<NC, WS>;
    constexpr int NW = Acc1<NC, WS>::NW, NQ = 2 * NC + NW;
    const int lane = threadIdx.x, ph = lane / kLW;
    double S[2 * NC], H[NW];
#pragma unroll
    for (int q = 0; q < 2 * NC; ++q) S[q] = 0.0;
#pragma unroll
    for (int q = 0; q < NW; ++q) H[q] = 0.0;
    const int CH = a.CH; // a multiple of kLP
    const int c_begin = wlo / CH, c_end = (whi + CH - 1) / CH;
    if (lane == 0) TL::issue(a, sm, c_begin, CH, &bar[0]);
    const size_t sw = (size_t)a.n_wp;
    const size_t cj = (size_t)a.n_m * 8 * sw;
    const int kbase = (int)a.k_min;
    const double df = a.df, h = (double)kLP * df, h2 = h * h, h3 = h2 * h;
    double ts4 = 0.0;
    if (a.t_shift) {
        const int w = a.perm[pw];
        if (w >= 0) ts4 = 4.0 * a.t_shift[(size_t)w * a.ts_stride];
    }
    // the interval's cubics of this lane's walker and the lane's recurrence state: they live across chunks
    double cA0 = 0, cA1 = 0, cA2 = 0, cA3 = 0, cP0 = 0, cP1 = 0, cP2 = 0, cP3 = 0, nxj = 0;
    double A = 0, d1A = 0, d2A = 0, d3A = 0, sz = 0, cz = 1, sw_ = 0, cw = 1, sv = 0, cv = 1, su = 0, cu = 1;
    int jl = -1, steps = kLaneSync; // rows since the last re-synchronisation
    for (int c = c_begin; c < c_end; ++c) {
        const int st = (c - c_begin) & 1;
        const uint32_t par = (uint32_t)((c - c_begin) >> 1) & 1u;
        if (lane == 0 && c + 1 < c_end) TL::issue(a, sm + (size_t)(st ^ 1) * CH * TL::DPB, c + 1, CH, &bar[st ^ 1]);
        mbar_wait(&bar[st], par);
        const double *sg = sm + (size_t)st * CH * TL::DPB;
        const int cb = c * CH;
        const double *sgc = sg - (size_t)cb * 2 * NC; // addressed by global bin
        const int ce = min(cb + CH, whi);
        int i = max(cb, wlo);
        while (i < ce) {
            while (j < a.n_nodes - 2 && __ldg(a.bstart + j + 1) <= i) ++j;
            const int j_end = (j < a.n_nodes - 2) ? __ldg(a.bstart + j + 1) : INT_MAX; // end of the interval
            const int seg_end = min(j_end, ce);
            if (j != jl) {
                const double *cc = a.C + (size_t)j * cj + pw;
                cA0 = cc[0]; cA1 = cc[sw]; cA2 = cc[2 * sw]; cA3 = cc[3 * sw];
                cP0 = cc[4 * sw]; cP1 = cc[5 * sw]; cP2 = cc[6 * sw]; cP3 = cc[7 * sw];
                const double xj = __ldg(a.xj + j);
                nxj = -xj;
                if (a.t_shift) { cP0 += qc_linear_mod_cycle(xj, ts4); cP1 += ts4; }
                // <h|h> of the walker's whole stretch in this interval, [m0, m1), from the weight moments
                const int m0 = max(i, lo), m1 = min(min(j_end, whi), hi);
                if (ph == 0 && m0 < m1) {
                    const bool first = m0 == __ldg(a.bstart + j);
                    const double q0 = cA0 * cA0, q1 = 2.0 * cA0 * cA1, q2 = fma(2.0 * cA0, cA2, cA1 * cA1);
                    const double q3 = 2.0 * fma(cA0, cA3, cA1 * cA2), q4 = fma(2.0 * cA1, cA3, cA2 * cA2);
                    const double q5 = 2.0 * cA2 * cA3, q6 = cA3 * cA3;
#pragma unroll
                    for (int r = 0; r < NW; ++r) {
                        const double *Q = a.wmom + (size_t)(r * 7) * a.n_f_pad;
                        auto mo = [&](int q) { return __ldg(Q + (size_t)q * a.n_f_pad + m1 - 1) - (first ? 0.0 : __ldg(Q + (size_t)q * a.n_f_pad + m0 - 1)); };
                        double hs = q0 * mo(0);
                        hs = fma(q1, mo(1), hs); hs = fma(q2, mo(2), hs); hs = fma(q3, mo(3), hs);
                        hs = fma(q4, mo(4), hs); hs = fma(q5, mo(5), hs); hs = fma(q6, mo(6), hs);
                        H[r] += hs;
                    }
                }
                d3A = 6.0 * cA3 * h3;
                LL_ROT_SINCOS(6.0 * cP3 * h3, su, cu);
                unit_modulus(cu, su);
                steps = kLaneSync; // forces a re-synchronisation below
                jl = j;
            }
            const int b0 = max(i, lo), b1 = min(seg_end, hi); // this lane's walker inside the stretch
            const int r_end = (seg_end - 1) / kLP;
            int r = i / kLP;
            while (r <= r_end) {
                if (steps >= kLaneSync) { // this lane's state at its bin of row r, from the cubics
                    const double t = fma((double)(kbase + kLP * r + ph), df, nxj);
                    const double tt = fma(2.0, t, h), q3 = fma(3.0 * t, t + h, h2), t1 = t + h;
                    A = fma(fma(fma(cA3, t, cA2), t, cA1), t, cA0);
                    d1A = h * fma(cA3, q3, fma(cA2, tt, cA1));
                    d2A = h2 * fma(6.0 * cA3, t1, 2.0 * cA2);
                    LL_ROT_SINCOS(fma(fma(fma(cP3, t, cP2), t, cP1), t, cP0), sz, cz);
                    LL_ROT_SINCOS(h * fma(cP3, q3, fma(cP2, tt, cP1)), sw_, cw);
                    LL_ROT_SINCOS(h2 * fma(6.0 * cP3, t1, 2.0 * cP2), sv, cv);
                    unit_modulus(cz, sz);
                    unit_modulus(cw, sw_);
                    unit_modulus(cv, sv);
                    steps = 0;
                }
                const int r1 = min(r_end, r + (kLaneSync - steps) - 1);
                steps += r1 - r + 1;
#pragma unroll 4
                for (; r <= r1; ++r) {
                    const int ii = kLP * r + ph;
                    const double Am = (ii >= b0 && ii < b1) ? A : 0.0;
                    const double u = Am * cz, v = Am * sz; // h = u - i v
                    double g[2 * NC];
                    load_g<NC>(sgc, ii, g);
#pragma unroll
                    for (int cch = 0; cch < NC; ++cch) {
                        S[2 * cch] = fma(g[2 * cch], u, S[2 * cch]); S[2 * cch] = fma(g[2 * cch + 1], v, S[2 * cch]);
                        S[2 * cch + 1] = fma(g[2 * cch + 1], u, S[2 * cch + 1]); S[2 * cch + 1] = fma(-g[2 * cch], v, S[2 * cch + 1]);
                    }
                    const double nzc = fma(cz, cw, -(sz * sw_)), nzs = fma(sz, cw, cz * sw_);
                    const double nwc = fma(cw, cv, -(sw_ * sv)), nws = fma(sw_, cv, cw * sv);
                    const double nvc = fma(cv, cu, -(sv * su)), nvs = fma(sv, cu, cv * su);
                    cz = nzc; sz = nzs; cw = nwc; sw_ = nws; cv = nvc; sv = nvs;
                    A += d1A; d1A += d2A; d2A += d3A;
                }
            }
            // a row that straddles the end of the interval is taken again by the next interval (complementary mask)
            i = seg_end;
        }
        poison_stage(sg, CH * TL::DPB);
        __syncthreads(); // (one warp) done with stage st before it is refilled two chunks later
    }
#pragma unroll
    for (int q = 0; q < 2 * NC; ++q)
#pragma unroll
        for (int o = kLW; o < 32; o <<= 1) S[q] += __shfl_xor_sync(0xffffffffu, S[q], o); // over the phases of a walker
    if (ph == 0) {
        double *o = a.part + (size_t)item * NQ * 32 + (pw & 31);
#pragma unroll
        for (int q = 0; q < 2 * NC; ++q) o[q * 32] = S[q];
#pragma unroll
        for (int q = 0; q < NW; ++q) o[(2 * NC + q) * 32] = H[q];
    }
}

// NM1 = 1: single-mode specialisation (NQ = 2 NC + NW partial sums per walker and tile); 0: any n_m (NQ = 2).
// SMALL = 1 (batches of up to 1024 walkers; blocks of ONE warp): block b is item b of the group table — bins
// [i0, i1) of one group of 32 walkers, an equal share of the batch's active bins — instead of (walker block, tile);
// its partial sums go to part[b][NQ][32].
template <int NM1, int NC, bool WS, int SMALL>
__global__ void __launch_bounds__(128, (NC == 2 && WS) ? (NM1 ? (SMALL ? LL_FUSED_MINB_SMALL : LL_FUSED_MINB) : 4) : ((NM1 && !SMALL) ? LL_FUSED_MINB_PC : 3))
k_full_fused(FusedArgs a)
{
    using TL = Tile<NC, WS>;
#ifndef LL_ROT_UNROLL_PC
#define LL_ROT_UNROLL_PC 2
#endif
#ifndef LL_ROT_UNROLL_MASKED
#define LL_ROT_UNROLL_MASKED 2
#endif
#ifndef LL_ROT_UNROLL_SMALL
#define LL_ROT_UNROLL_SMALL 4 // 160 walkers on the config-2 grid: 1: 0.156 ms, 2: 0.151, 3: 0.150, 4: 0.148
#endif
    constexpr int UR = SMALL ? LL_ROT_UNROLL_SMALL : ((NC == 2 && WS) ? kRotUnroll : LL_ROT_UNROLL_PC); // trip length of the unmasked recurrence loop
    extern __shared__ __align__(128) double sm[];
    __shared__ __align__(8) uint64_t bar[2];
    __shared__ int s_lo, s_hi;

    const int tid = threadIdx.x;
    int p, tile, i0, i1, j_hint = 0;
    bool lanes_item = false;
    if (SMALL) {
        tile = blockIdx.x;
        if (tile >= __ldg(a.grp_tab + 32)) return;
        const int *it = a.grp_tab + grp_off_items() + tile;
        const int mi = gridDim.x; // the table's row length = the grid
        i0 = __ldg(it + mi);
        i1 = __ldg(it + 2 * mi);
        j_hint = __ldg(it + 3 * mi);
        const int code = __ldg(it);
        lanes_item = NM1 && LL_SMALL_LANES && code < 0; // kLW walkers from sorted position -code - 1 on, lanes = (walker, phase)
        p = lanes_item ? (-code - 1) + tid % kLW : code * 32 + tid;
    } else {
        p = blockIdx.x * blockDim.x + tid;
        tile = blockIdx.y;
        i0 = __ldg(a.tile_start + tile);
        i1 = __ldg(a.tile_start + tile + 1); // tile = dense bins [i0, i1)
    }
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
    if (blo >= bhi) { // no walker of this block has bins in this tile
        if (SMALL) {  // an item of the cost partition may hold no bin at all, and k_finalize_small does read it
            constexpr int NQ0 = NM1 ? 2 * NC + Acc1<NC, WS>::NW : 2;
#pragma unroll
            for (int q = 0; q < NQ0; ++q) a.part[((size_t)tile * NQ0 + q) * 32 + tid] = 0.0;
        }
        return; // large batches: k_finalize never reads it
    }

    if (SMALL && NM1 && LL_SMALL_LANES && lanes_item) {
        fused_lanes_item<NC, WS>(a, p, lo, hi, blo, bhi, j_hint, tile, sm, bar);
        return;
    }
    const int CH = a.CH;
    const int c_begin = blo / CH, c_end = (bhi + CH - 1) / CH;
    if (tid == 0) TL::issue(a, sm, c_begin, CH, &bar[0]);

    const size_t sw = (size_t)a.n_wp;
    const size_t cj = (size_t)a.n_m * 8 * sw;
    int j = SMALL ? j_hint : find_interval_of_bin(a.bstart, a.n_nodes, blo); // the bin loop moves a hint up to its interval
    int jl = -1;
    double cA0 = 0, cA1 = 0, cA2 = 0, cA3 = 0, cP0 = 0, cP1 = 0, cP2 = 0, cP3 = 0, nxj = 0;
    const int kbase = (int)a.k_min; // k_min + n_f < 2^31 is checked on the host
    double ts4 = 0.0;               // 4 t_shift: the linear phase term in quarter cycles per Hz
    if (a.t_shift) {
        const int w = a.perm[p];
        if (w >= 0) ts4 = 4.0 * a.t_shift[(size_t)w * a.ts_stride];
    }
    Acc1<NC, WS> acc; // NM1: S^c, H;  generic: S[0] = d_h, S[1] = h_h
    acc.zero();

    for (int c = c_begin; c < c_end; ++c) {
        const int st = (c - c_begin) & 1;
        const uint32_t ph = (uint32_t)((c - c_begin) >> 1) & 1u;
        if (tid == 0 && c + 1 < c_end) TL::issue(a, sm + (size_t)(st ^ 1) * CH * TL::DPB, c + 1, CH, &bar[st ^ 1]);
        mbar_wait(&bar[st], ph);
        const double *sg = sm + (size_t)st * CH * TL::DPB;
        const int cb = c * CH;
        const double *sgc = sg - (size_t)cb * 2 * NC;      // addressed by global bin
        const double *sWc = sg + (size_t)CH * 2 * NC - cb; // weight row r of bin ii: sWc[r CH + ii]
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
                        const double xj = __ldg(a.xj + j);
                        nxj = -xj;
                        if (a.t_shift) { cP0 += qc_linear_mod_cycle(xj, ts4); cP1 += ts4; }
                        jl = j;
                    }
                    // bins every lane of the warp has inside its band run without the per-lane mask
                    const int flo = __reduce_max_sync(0xffffffffu, max(lo, i));
                    const int fhi = __reduce_min_sync(0xffffffffu, min(hi, seg_end));
                    // masked stretch [b0, b1): by recurrence with the mask when it is long enough, else bin by bin
                    auto masked = [&](int b0, int b1) {
                        if (LL_FUSED_ROT && b1 - b0 >= 8)
                            fused_bins_rot<true, NC, WS, true, LL_ROT_UNROLL_MASKED>(b0, b1, tlo, thi, kbase, a.df, nxj, cA0, cA1, cA2, cA3,
                                                                                     cP0, cP1, cP2, cP3, sgc, sWc, CH, acc);
                        else
                            fused_bins_nm1<true, NC, WS>(b0, b1, tlo, thi, kbase, a.df, nxj, cA0, cA1, cA2, cA3, cP0, cP1, cP2, cP3,
                                                         sgc, sWc, CH, acc);
                    };
                    if (flo < fhi) {
                        masked(wlo, flo);
                        if (LL_FUSED_ROT && fhi - flo >= 8) {
                            if (LL_H_MOMENTS && a.wmom) {
                                // sum_k W^r_k A(t_k)^2 over the stretch from the weight moments (two of the 27 slots per bin; 1 + NC
                                // of the 33 with per-channel rows): A^2 = sum_p q_p t^p, M^r_p = sum_k W^r_k t_k^p = difference of two
                                // prefix entries
                                constexpr int NWR = Acc1<NC, WS>::NW;
                                double mo[NWR][7];
                                const bool first = flo == __ldg(a.bstart + j);
#pragma unroll
                                for (int r = 0; r < NWR; ++r)
#pragma unroll
                                    for (int q = 0; q < 7; ++q) {
                                        const double *Q = a.wmom + (size_t)(r * 7 + q) * a.n_f_pad;
                                        mo[r][q] = __ldg(Q + fhi - 1) - (first ? 0.0 : __ldg(Q + flo - 1));
                                    }
                                fused_bins_rot<false, NC, WS, false, UR>(flo, fhi, tlo, thi, kbase, a.df, nxj, cA0, cA1, cA2, cA3, cP0,
                                                                     cP1, cP2, cP3, sgc, sWc, CH, acc);
                                const double q0 = cA0 * cA0, q1 = 2.0 * cA0 * cA1, q2 = fma(2.0 * cA0, cA2, cA1 * cA1);
                                const double q3 = 2.0 * fma(cA0, cA3, cA1 * cA2), q4 = fma(2.0 * cA1, cA3, cA2 * cA2);
                                const double q5 = 2.0 * cA2 * cA3, q6 = cA3 * cA3;
#pragma unroll
                                for (int r = 0; r < NWR; ++r) {
                                    double hs = q0 * mo[r][0];
                                    hs = fma(q1, mo[r][1], hs);
                                    hs = fma(q2, mo[r][2], hs);
                                    hs = fma(q3, mo[r][3], hs);
                                    hs = fma(q4, mo[r][4], hs);
                                    hs = fma(q5, mo[r][5], hs);
                                    hs = fma(q6, mo[r][6], hs);
                                    acc.H[r] += hs;
                                }
                            } else {
                                fused_bins_rot<false, NC, WS, true, UR>(flo, fhi, tlo, thi, kbase, a.df, nxj, cA0, cA1,
                                                                                          cA2, cA3, cP0, cP1, cP2, cP3, sgc, sWc, CH, acc);
                            }
                        } else
                            fused_bins_nm1<false, NC, WS>(flo, fhi, tlo, thi, kbase, a.df, nxj, cA0, cA1, cA2, cA3, cP0, cP1,
                                                          cP2, cP3, sgc, sWc, CH, acc);
                        masked(fhi, whi);
                    } else {
                        masked(wlo, whi);
                    }
                } else {
                    // any number of modes: chunks of four bins with the MODE loop outside the bins, so that a mode's
                    // 8 coefficients and 2 NC transfer factors are read once per chunk (not once per bin) and the four
                    // bins are four independent cubic -> sincos -> T^c h chains in flight per thread
                    const double xj = __ldg(a.xj + j);
                    nxj = -xj;
                    const double sh0 = a.t_shift ? qc_linear_mod_cycle(xj, ts4) : 0.0;
                    const double *cc0 = a.C + (size_t)j * cj + p;
                    for (int c4 = wlo; c4 < whi; c4 += 4) {
                        double t4[4], h4[4][2 * NC];
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            t4[k] = fma((double)(kbase + c4 + k), a.df, nxj);
#pragma unroll
                            for (int q = 0; q < 2 * NC; ++q) h4[k][q] = 0.0;
                        }
#pragma unroll 1
                        for (int m = 0; m < a.n_m; ++m) {
                            const double *cc = cc0 + (size_t)m * 8 * sw;
                            double co[8];
#pragma unroll
                            for (int q = 0; q < 8; ++q) co[q] = cc[(size_t)q * sw];
                            if (a.t_shift) { co[4] += sh0; co[5] += ts4; }
                            const double *tfp = a.TF + (size_t)m * 2 * NC * sw + p;
                            double tf[2 * NC];
#pragma unroll
                            for (int q = 0; q < 2 * NC; ++q) tf[q] = tfp[(size_t)q * sw];
#pragma unroll
                            for (int k = 0; k < 4; ++k) {
                                const double A = fma(fma(fma(co[3], t4[k], co[2]), t4[k], co[1]), t4[k], co[0]);
                                const double y = fma(fma(fma(co[7], t4[k], co[6]), t4[k], co[5]), t4[k], co[4]);
                                double u, v; // h_m = u - i v
                                amp_expi_qc(A, y, u, v);
                                apply_tf<NC>(tf, u, v, h4[k]);
                            }
                        }
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            const int ii = c4 + k;
                            if (ii < whi && ii >= tlo && ii < thi) accumulate_bin<NC, WS>(sgc, sWc, CH, ii, h4[k], acc.S[0], acc.S[1]);
                        }
                    }
                }
            }
            i = seg_end;
        }
        poison_stage(sg, CH * TL::DPB);
        __syncthreads(); // everyone is done with stage st before it is refilled two chunks later
    }
    constexpr int NQ = NM1 ? 2 * NC + Acc1<NC, WS>::NW : 2;
    const size_t so = SMALL ? 32 : sw; // stride between the partial sums of one record
    double *o = SMALL ? a.part + (size_t)tile * NQ * 32 + tid : a.part + ((size_t)tile * NQ) * sw + p;
    if (NM1) {
#pragma unroll
        for (int q = 0; q < 2 * NC; ++q) o[(size_t)q * so] = acc.S[q];
#pragma unroll
        for (int q = 0; q < Acc1<NC, WS>::NW; ++q) o[(size_t)(2 * NC + q) * so] = acc.H[q];
    } else {
        o[0] = acc.S[0]; o[so] = acc.S[1];
    }
}

// ---------------------------------------------------------------------------------------------------
// F3 for several modes, large batches, by the rotation recurrence (the paper's higher-mode analysis ran this brute-force
// likelihood).  k_full_fused<0> evaluates every (bin, mode) directly: two cubics and a sincos, 37 FP64
// instructions + T^c h.  Here every mode carries its own recurrence state (z, w, v and the amplitude with its two
// differences: 9 doubles in registers per mode), exactly as fused_bins_rot does for one mode: per (bin, mode) 12
// (rotations) + 3 (amplitude) + 2 (A z) + 4 NC (T^c h) = 25 for two channels, plus per bin Re(g^c h^c) and W |h^c|^2.  What
// is constant inside a re-synchronisation stretch — u = e^{i D3 Psi}, D3 A, T^c_m: 3 + 2 NC doubles per mode — lives in
// shared memory (per thread, [q][thread]: conflict-free).  The modes are NM independent chains per bin, so a thread has
// plenty of instruction-level parallelism although only three blocks fit an SM.  Same mapping, staging, tiles and band
// logic as k_full_fused; bins outside a lane's band advance the recurrence but are not accumulated.
// ---------------------------------------------------------------------------------------------------
#ifndef LL_HM_MINB
#define LL_HM_MINB 2 // six modes keep 54 doubles of recurrence state: at three blocks per SM (168 registers) the bin loop spills and the kernel takes 36.5 ms at config-2 size with 2048 walkers; at two (255 registers) 16.4 ms (direct route: 24.2 ms)
#endif
#ifndef LL_HM_UNROLL
#define LL_HM_UNROLL 1
#endif
constexpr int kHmUnroll = LL_HM_UNROLL;
// SMALL = 1: one-warp blocks over the planner's group items (batches below 384 walkers), as k_full_fused<.., SMALL = 1>.
template <int NM, int NC, bool WS, int SMALL = 0>
__global__ void __launch_bounds__(128, LL_HM_MINB) k_full_fused_hm(FusedArgs a)
{
    using TL = Tile<NC, WS>;
    constexpr int NK = 3 + 2 * NC; // constants per mode in shared memory: cu, su, d3A, T^c (re, im)
    extern __shared__ __align__(128) double sm[];
    __shared__ __align__(8) uint64_t bar[2];
    __shared__ int s_lo, s_hi;
    const int tid = threadIdx.x, nthr = blockDim.x;
    int p, tile, i0, i1, j_hint = 0;
    if (SMALL) {
        tile = blockIdx.x;
        if (tile >= __ldg(a.grp_tab + 32)) return;
        const int *it = a.grp_tab + grp_off_items() + tile;
        const int mi = gridDim.x;
        i0 = __ldg(it + mi);
        i1 = __ldg(it + 2 * mi);
        j_hint = __ldg(it + 3 * mi);
        p = __ldg(it) * 32 + tid;
    } else {
        p = blockIdx.x * blockDim.x + tid;
        tile = blockIdx.y;
        i0 = __ldg(a.tile_start + tile);
        i1 = __ldg(a.tile_start + tile + 1);
    }
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
    if (blo >= bhi) { // k_finalize never reads a tile no walker of the block touches; F4 of the small route reads every item
        if (SMALL) { a.part[((size_t)tile * 2) * 32 + tid] = 0.0; a.part[((size_t)tile * 2 + 1) * 32 + tid] = 0.0; }
        return;
    }

    const int CH = a.CH;
    double *kst = sm + (size_t)2 * CH * TL::DPB + tid; // this thread's constants: kst[(m * NK + q) * nthr]
    const int c_begin = blo / CH, c_end = (bhi + CH - 1) / CH;
    if (tid == 0) TL::issue(a, sm, c_begin, CH, &bar[0]);
    const size_t sw = (size_t)a.n_wp;
    const size_t cj = (size_t)a.n_m * 8 * sw;
    const int kbase = (int)a.k_min;
    const double df = a.df, df2 = df * df, df3 = df2 * df;
    double ts4 = 0.0;
    if (a.t_shift) {
        const int w = a.perm[p];
        if (w >= 0) ts4 = 4.0 * a.t_shift[(size_t)w * a.ts_stride];
    }
    int j = SMALL ? j_hint : find_interval_of_bin(a.bstart, a.n_nodes, blo);
    int jl = -1, steps = kRotSync, expect = -1;
    double cz[NM], sz[NM], cw[NM], sw_[NM], cv[NM], sv[NM], A[NM], d1A[NM], d2A[NM];
#pragma unroll
    for (int m = 0; m < NM; ++m) { cz[m] = 1; sz[m] = 0; cw[m] = 1; sw_[m] = 0; cv[m] = 1; sv[m] = 0; A[m] = 0; d1A[m] = 0; d2A[m] = 0; }
    double s_dh = 0.0, s_hh = 0.0;

    for (int c = c_begin; c < c_end; ++c) {
        const int st = (c - c_begin) & 1;
        const uint32_t ph = (uint32_t)((c - c_begin) >> 1) & 1u;
        if (tid == 0 && c + 1 < c_end) TL::issue(a, sm + (size_t)(st ^ 1) * CH * TL::DPB, c + 1, CH, &bar[st ^ 1]);
        mbar_wait(&bar[st], ph);
        const double *sg = sm + (size_t)st * CH * TL::DPB;
        const int cb = c * CH;
        const double *sgc = sg - (size_t)cb * 2 * NC;
        const double *sWc = sg + (size_t)CH * 2 * NC - cb;
        const int ce = min(cb + CH, bhi);
        int i = max(cb, blo);
        while (i < ce) {
            while (j < a.n_nodes - 2 && __ldg(a.bstart + j + 1) <= i) ++j;
            const int seg_end = (j < a.n_nodes - 2) ? min(__ldg(a.bstart + j + 1), ce) : ce;
            int tlo = max(i, lo), thi = min(seg_end, hi);
            if (tlo >= thi) { tlo = INT_MAX; thi = INT_MIN; }
            const int wlo = __reduce_min_sync(0xffffffffu, tlo);
            const int whi = __reduce_max_sync(0xffffffffu, thi);
            if (j != jl) { steps = kRotSync; jl = j; } // a new interval: re-synchronise at its first bin
            if (wlo != expect) steps = kRotSync;       // the warp's bins are not contiguous with the last stretch
            int ii = wlo;
            while (ii < whi) {
                if (steps >= kRotSync) { // every mode's state at bin ii, from its cubics
                    const double nxj = -__ldg(a.xj + j);
                    const double sh0 = a.t_shift ? qc_linear_mod_cycle(-nxj, ts4) : 0.0;
                    const double t = fma((double)(kbase + ii), df, nxj);
                    const double tt = fma(2.0, t, df), q3 = fma(3.0 * t, t + df, df2), t1 = t + df;
                    const double *cc0 = a.C + (size_t)j * cj + p;
#pragma unroll
                    for (int m = 0; m < NM; ++m) {
                        const double *cc = cc0 + (size_t)m * 8 * sw;
                        const double cA0 = cc[0], cA1 = cc[sw], cA2 = cc[2 * sw], cA3 = cc[3 * sw];
                        const double cP0 = cc[4 * sw] + sh0, cP1 = cc[5 * sw] + ts4, cP2 = cc[6 * sw], cP3 = cc[7 * sw];
                        A[m] = fma(fma(fma(cA3, t, cA2), t, cA1), t, cA0);
                        d1A[m] = df * fma(cA3, q3, fma(cA2, tt, cA1));
                        d2A[m] = df2 * fma(6.0 * cA3, t1, 2.0 * cA2);
                        double su, cu;
                        LL_ROT_SINCOS(fma(fma(fma(cP3, t, cP2), t, cP1), t, cP0), sz[m], cz[m]);
                        LL_ROT_SINCOS(df * fma(cP3, q3, fma(cP2, tt, cP1)), sw_[m], cw[m]);
                        LL_ROT_SINCOS(df2 * fma(6.0 * cP3, t1, 2.0 * cP2), sv[m], cv[m]);
                        LL_ROT_SINCOS(6.0 * cP3 * df3, su, cu);
                        unit_modulus(cz[m], sz[m]);
                        unit_modulus(cw[m], sw_[m]);
                        unit_modulus(cv[m], sv[m]);
                        unit_modulus(cu, su);
                        double *k = kst + (size_t)(m * NK) * nthr;
                        k[0] = cu; k[nthr] = su; k[2 * nthr] = 6.0 * cA3 * df3;
                        const double *tfp = a.TF + (size_t)m * 2 * NC * sw + p;
#pragma unroll
                        for (int q = 0; q < 2 * NC; ++q) k[(3 + q) * nthr] = tfp[(size_t)q * sw];
                    }
                    steps = 0;
                }
                const int ie = min(whi, ii + (kRotSync - steps));
                steps += ie - ii;
#pragma unroll kHmUnroll
                for (; ii < ie; ++ii) {
                    double h[2 * NC];
#pragma unroll
                    for (int q = 0; q < 2 * NC; ++q) h[q] = 0.0;
#pragma unroll
                    for (int m = 0; m < NM; ++m) {
                        const double *k = kst + (size_t)(m * NK) * nthr;
                        const double u = A[m] * cz[m], v = A[m] * sz[m]; // h_m = u - i v
#pragma unroll
                        for (int cch = 0; cch < NC; ++cch) {
                            const double tr = k[(3 + 2 * cch) * nthr], ti = k[(4 + 2 * cch) * nthr];
                            h[2 * cch] = fma(tr, u, h[2 * cch]); h[2 * cch] = fma(ti, v, h[2 * cch]);
                            h[2 * cch + 1] = fma(ti, u, h[2 * cch + 1]); h[2 * cch + 1] = fma(-tr, v, h[2 * cch + 1]);
                        }
                        const double cu = k[0], su = k[nthr];
                        const double nzc = fma(cz[m], cw[m], -(sz[m] * sw_[m])), nzs = fma(sz[m], cw[m], cz[m] * sw_[m]);
                        const double nwc = fma(cw[m], cv[m], -(sw_[m] * sv[m])), nws = fma(sw_[m], cv[m], cw[m] * sv[m]);
                        const double nvc = fma(cv[m], cu, -(sv[m] * su)), nvs = fma(sv[m], cu, cv[m] * su);
                        cz[m] = nzc; sz[m] = nzs; cw[m] = nwc; sw_[m] = nws; cv[m] = nvc; sv[m] = nvs;
                        A[m] += d1A[m]; d1A[m] += d2A[m]; d2A[m] += k[2 * nthr];
                    }
                    if (ii >= tlo && ii < thi) accumulate_bin<NC, WS>(sgc, sWc, CH, ii, h, s_dh, s_hh);
                }
            }
            if (wlo < whi) expect = whi;
            i = seg_end;
        }
        poison_stage(sg, CH * TL::DPB);
        __syncthreads();
    }
    if (SMALL) {
        a.part[((size_t)tile * 2) * 32 + tid] = s_dh;
        a.part[((size_t)tile * 2 + 1) * 32 + tid] = s_hh;
        return;
    }
    double *o = a.part + ((size_t)tile * 2) * sw + p;
    o[0] = s_dh; o[sw] = s_hh;
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
#ifndef LL_MIXED_ROT
#define LL_MIXED_ROT 0 // 1: the phase by the FP64 rotation recurrence, the rest in binary32 (fused_pairs_rot_mixed).  Measured at
                       // config 2 (ncu r02, profiles/r02_full_fused_mixed_cfg2.md): 9.6 ms against 9.98 ms for the direct
                       // binary32 sincos route and 10.8 ms for the FP64 kernel, FP64 pipe 50 % busy, XU pipe 40 % busy —
                       // the three FP64 -> binary32 conversions per bin (cos, sin, W A^2 hand-off) run on the XU pipe at a
                       // quarter of the FP64 rate and stall dispatch — and max |delta log L| 1.07e-3 against FP64, over
                       // the 1e-3 bar.  Off: the variant cannot pay on this chip.
#endif

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

// The same pairs with the phase advanced by the FP64 rotation recurrence of fused_bins_rot (z <- z w, w <- w v,
// v <- v u: 12 FP64 instructions per bin, re-synchronised every kRotSync bins) and everything else in binary32:
// the amplitude as its Taylor cubic around the re-sync point (the offset is at most 32 bins, so the binary32 rounding
// is relative to A itself and not cumulative), A e^{-i Psi}, the MACs with the binary32 data tile and W A^2, two bins
// per f32x2 instruction, partial sums of 8 terms per accumulator lane flushed into the FP64 accumulators.
// The FP64 pipe carries 12 of the FP64 kernel's 27 instructions per bin.
__device__ __forceinline__ void fused_pairs_rot_mixed(int b0, int b1, int kbase, double df, double nxj, double cA0, double cA1,
                                                      double cA2, double cA3, double cP0, double cP1, double cP2, double cP3,
                                                      const float *__restrict__ sgp, const double *__restrict__ sWc,
                                                      MixedAcc &acc)
{
    const double df2 = df * df, df3 = df2 * df;
    const float dff = __double2float_rn(df);
    double su, cu;
    LL_ROT_SINCOS(6.0 * cP3 * df3, su, cu);
    unit_modulus(cu, su);
    const f32x2 dS = pack2(2.0f * dff, 2.0f * dff), one2 = pack2(1.0f, 1.0f);
    for (int k0 = b0; k0 < b1; k0 += kRotSync) {
        const int k1 = min(k0 + kRotSync, b1);
        const double t = fma((double)(kbase + k0), df, nxj);
        const double tt = fma(2.0, t, df), q3 = fma(3.0 * t, t + df, df2), t1 = t + df;
        // amplitude: Taylor coefficients at t, in binary32
        const float a0 = __double2float_rn(fma(fma(fma(cA3, t, cA2), t, cA1), t, cA0));
        const float a1 = __double2float_rn(fma(fma(3.0 * cA3, t, 2.0 * cA2), t, cA1));
        const float a2 = __double2float_rn(fma(3.0 * cA3, t, cA2));
        const float a3 = __double2float_rn(cA3);
        const f32x2 A0 = pack2(a0, a0), A1 = pack2(a1, a1), A2 = pack2(a2, a2), A3 = pack2(a3, a3);
        double sz, cz, sw, cw, sv, cv;
        LL_ROT_SINCOS(fma(fma(fma(cP3, t, cP2), t, cP1), t, cP0), sz, cz);
        LL_ROT_SINCOS(df * fma(cP3, q3, fma(cP2, tt, cP1)), sw, cw);
        LL_ROT_SINCOS(df2 * fma(6.0 * cP3, t1, 2.0 * cP2), sv, cv);
        unit_modulus(cz, sz);
        unit_modulus(cw, sw);
        unit_modulus(cv, sv);
        f32x2 S = pack2(0.0f, dff); // offsets of the pair's two bins from the re-sync point
        for (int base = k0; base < k1; base += 2 * kMixedChain) {
            const int end = min(base + 2 * kMixedChain, k1);
            f32x2 aXU = 0, aYV = 0, aYU = 0, aXV = 0, eXU = 0, eYV = 0, eYU = 0, eXV = 0; // +0.0f in both lanes
#pragma unroll 2
            for (int ii = base; ii < end; ii += 2) {
                const float c0 = __double2float_rn(cz), s0 = __double2float_rn(sz);
                double nzc = fma(cz, cw, -(sz * sw)), nzs = fma(sz, cw, cz * sw);
                double nwc = fma(cw, cv, -(sw * sv)), nws = fma(sw, cv, cw * sv);
                double nvc = fma(cv, cu, -(sv * su)), nvs = fma(sv, cu, cv * su);
                cz = nzc; sz = nzs; cw = nwc; sw = nws; cv = nvc; sv = nvs;
                const float c1 = __double2float_rn(cz), s1 = __double2float_rn(sz);
                nzc = fma(cz, cw, -(sz * sw)); nzs = fma(sz, cw, cz * sw);
                nwc = fma(cw, cv, -(sw * sv)); nws = fma(sw, cv, cw * sv);
                nvc = fma(cv, cu, -(sv * su)); nvs = fma(sv, cu, cv * su);
                cz = nzc; sz = nzs; cw = nwc; sw = nws; cv = nvc; sv = nvs;
                const f32x2 Af = fma2(fma2(fma2(A3, S, A2), S, A1), S, A0);
                S = fma2(dS, one2, S);
                const f32x2 U = mul2(Af, pack2(c0, c1)), V = mul2(Af, pack2(s0, s1)); // h = u - i v per lane
                const ulonglong2 gA = *reinterpret_cast<const ulonglong2 *>(sgp + (ii >> 1) * 8);
                const ulonglong2 gE = *reinterpret_cast<const ulonglong2 *>(sgp + (ii >> 1) * 8 + 4);
                aXU = fma2(gA.x, U, aXU); aYV = fma2(gA.y, V, aYV); aYU = fma2(gA.y, U, aYU); aXV = fma2(gA.x, V, aXV);
                eXU = fma2(gE.x, U, eXU); eYV = fma2(gE.y, V, eYV); eYU = fma2(gE.y, U, eYU); eXV = fma2(gE.x, V, eXV);
                // <h|h> = sum W A^2 stays in FP64 (all terms positive: binary32 sums lose ~1e-8 of 2.5e5, reading R15)
                const double2 w = *reinterpret_cast<const double2 *>(sWc + ii);
                float al, ah;
                unpack2(Af, al, ah);
                const double ald = (double)al, ahd = (double)ah;
                acc.sH = fma(w.x * ald, ald, acc.sH);
                acc.sH = fma(w.y * ahd, ahd, acc.sH);
            }
            float l0, h0, l1, h1;
            unpack2(aXU, l0, h0); unpack2(aYV, l1, h1); acc.sAr += (double)((l0 + h0) + (l1 + h1));
            unpack2(aYU, l0, h0); unpack2(aXV, l1, h1); acc.sAi += (double)((l0 + h0) - (l1 + h1));
            unpack2(eXU, l0, h0); unpack2(eYV, l1, h1); acc.sEr += (double)((l0 + h0) + (l1 + h1));
            unpack2(eYU, l0, h0); unpack2(eXV, l1, h1); acc.sEi += (double)((l0 + h0) - (l1 + h1));
        }
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
    double ts4 = 0.0; // 4 t_shift (reading R32), folded into the phase cubic of the current interval
    if (a.t_shift) {
        const int w = a.perm[p];
        if (w >= 0) ts4 = 4.0 * a.t_shift[(size_t)w * a.ts_stride];
    }
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
                    const double xj = __ldg(a.xj + j);
                    nxj = -xj;
                    if (a.t_shift) { cP0 += qc_linear_mod_cycle(xj, ts4); cP1 += ts4; }
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
                    if (LL_MIXED_ROT && phi - plo >= 16)
                        fused_pairs_rot_mixed(plo, phi, kbase, a.df, nxj, cA0, cA1, cA2, cA3, cP0, cP1, cP2, cP3, sgp, sWc, acc);
                    else
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
        poison_stage(sg, CH * 3);
        __syncthreads();
    }
    double *o = a.part + ((size_t)tile * 5) * sw + p;
    o[0] = acc.sAr; o[sw] = acc.sAi; o[2 * sw] = acc.sEr; o[3 * sw] = acc.sEi; o[4 * sw] = acc.sH;
}

// ---------------------------------------------------------------------------------------------------
// F3 with a frequency-dependent transfer function (Eq. 8-9).  Same mapping, staging and
// band logic as k_full_fused; per (walker, bin, mode) 2 + 2 NC cubics (amplitude, phase, Re/Im of every T^c), then
// h^c += T^c(f) A e^{-i Psi}.  Coefficient block per (interval, mode): 8 + 8 NC doubles, walker fastest.
// NM1 = 1: the coefficients of the current interval live in registers; 0: any n_m, coefficients re-read per
// chunk of bins through L1 (they would not fit in registers for several modes).
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ double cubic4(const double *c4, double t)
{
    return fma(fma(fma(c4[3], t, c4[2]), t, c4[1]), t, c4[0]);
}

#ifndef LL_TF_MINB
#define LL_TF_MINB 5 // config-2 size, one mode: 3 blocks per SM (153 registers) 17.33 ms, 4 (128) 17.78, 5 (96, spills outside the bin loop) 16.90, 6 (80) 17.58
#endif
// A lanes item (fused_lanes_item above) of the T(f) kernel, single mode: lane = (walker, bin phase); A e^{-i Psi} by the lane's
// own stride-kLP recurrence, the four T cubics by Horner at the lane's bin, T^c h, Re(g^c h^c) and W |h^c|^2 per row (with T(f)
// there is no moment form of <h|h>).  The walker's 8 + 8 NC coefficients of the current interval live in registers.
template <int NC, bool WS>
__device__ __forceinline__ void fused_lanes_item_tf(const FusedArgs &a, int pw, int lo, int hi, int wlo, int whi, int j, int item,
                                                    double *sm, uint64_t *bar)
{
    using TL = Tile<NC, WS>;
    constexpr int NCO = 8 + 8 * NC;
    const int lane = threadIdx.x, ph = lane / kLW;
    double s_dh = 0.0, s_hh = 0.0;
    const int CH = a.CH;
    const int c_begin = wlo / CH, c_end = (whi + CH - 1) / CH;
    if (lane == 0) TL::issue(a, sm, c_begin, CH, &bar[0]);
    const size_t sw = (size_t)a.n_wp;
    const size_t cj = (size_t)a.n_m * NCO * sw;
    const int kbase = (int)a.k_min;
    const double df = a.df, h = (double)kLP * df, h2 = h * h, h3 = h2 * h;
    double ts4 = 0.0;
    if (a.t_shift) {
        const int w = a.perm[pw];
        if (w >= 0) ts4 = 4.0 * a.t_shift[(size_t)w * a.ts_stride];
    }
    double co[NCO], nxj = 0;
    double A = 0, d1A = 0, d2A = 0, d3A = 0, sz = 0, cz = 1, sw_ = 0, cw = 1, sv = 0, cv = 1, su = 0, cu = 1;
    int jl = -1, steps = kLaneSync;
    for (int c = c_begin; c < c_end; ++c) {
        const int st = (c - c_begin) & 1;
        const uint32_t par = (uint32_t)((c - c_begin) >> 1) & 1u;
        if (lane == 0 && c + 1 < c_end) TL::issue(a, sm + (size_t)(st ^ 1) * CH * TL::DPB, c + 1, CH, &bar[st ^ 1]);
        mbar_wait(&bar[st], par);
        const double *sg = sm + (size_t)st * CH * TL::DPB;
        const int cb = c * CH;
        const double *sgc = sg - (size_t)cb * 2 * NC;
        const double *sWc = sg + (size_t)CH * 2 * NC - cb;
        const int ce = min(cb + CH, whi);
        int i = max(cb, wlo);
        while (i < ce) {
            while (j < a.n_nodes - 2 && __ldg(a.bstart + j + 1) <= i) ++j;
            const int seg_end = (j < a.n_nodes - 2) ? min(__ldg(a.bstart + j + 1), ce) : ce;
            if (j != jl) {
                const double *cc = a.C + (size_t)j * cj + pw;
#pragma unroll
                for (int q = 0; q < NCO; ++q) co[q] = cc[(size_t)q * sw];
                const double xj = __ldg(a.xj + j);
                nxj = -xj;
                if (a.t_shift) { co[4] += qc_linear_mod_cycle(xj, ts4); co[5] += ts4; }
                d3A = 6.0 * co[3] * h3;
                LL_ROT_SINCOS(6.0 * co[7] * h3, su, cu);
                unit_modulus(cu, su);
                steps = kLaneSync;
                jl = j;
            }
            const int b0 = max(i, lo), b1 = min(seg_end, hi);
            const int r_end = (seg_end - 1) / kLP;
            int r = i / kLP;
            while (r <= r_end) {
                if (steps >= kLaneSync) {
                    const double t = fma((double)(kbase + kLP * r + ph), df, nxj);
                    const double tt = fma(2.0, t, h), q3 = fma(3.0 * t, t + h, h2), t1 = t + h;
                    A = cubic4(co, t);
                    d1A = h * fma(co[3], q3, fma(co[2], tt, co[1]));
                    d2A = h2 * fma(6.0 * co[3], t1, 2.0 * co[2]);
                    LL_ROT_SINCOS(cubic4(co + 4, t), sz, cz);
                    LL_ROT_SINCOS(h * fma(co[7], q3, fma(co[6], tt, co[5])), sw_, cw);
                    LL_ROT_SINCOS(h2 * fma(6.0 * co[7], t1, 2.0 * co[6]), sv, cv);
                    unit_modulus(cz, sz);
                    unit_modulus(cw, sw_);
                    unit_modulus(cv, sv);
                    steps = 0;
                }
                const int r1 = min(r_end, r + (kLaneSync - steps) - 1);
                steps += r1 - r + 1;
#pragma unroll 2
                for (; r <= r1; ++r) {
                    const int ii = kLP * r + ph;
                    const double t = fma((double)(kbase + ii), df, nxj);
                    const double u = A * cz, v = A * sz; // h = u - i v
                    double hc[2 * NC];
#pragma unroll
                    for (int cch = 0; cch < NC; ++cch) {
                        const double tr = cubic4(co + 8 + 8 * cch, t), ti = cubic4(co + 12 + 8 * cch, t);
                        hc[2 * cch] = fma(tr, u, ti * v);
                        hc[2 * cch + 1] = fma(ti, u, -(tr * v));
                    }
                    if (ii >= b0 && ii < b1) accumulate_bin<NC, WS>(sgc, sWc, CH, ii, hc, s_dh, s_hh);
                    const double nzc = fma(cz, cw, -(sz * sw_)), nzs = fma(sz, cw, cz * sw_);
                    const double nwc = fma(cw, cv, -(sw_ * sv)), nws = fma(sw_, cv, cw * sv);
                    const double nvc = fma(cv, cu, -(sv * su)), nvs = fma(sv, cu, cv * su);
                    cz = nzc; sz = nzs; cw = nwc; sw_ = nws; cv = nvc; sv = nvs;
                    A += d1A; d1A += d2A; d2A += d3A;
                }
            }
            i = seg_end;
        }
        poison_stage(sg, CH * TL::DPB);
        __syncthreads();
    }
#pragma unroll
    for (int o = kLW; o < 32; o <<= 1) { // over the phases of a walker
        s_dh += __shfl_xor_sync(0xffffffffu, s_dh, o);
        s_hh += __shfl_xor_sync(0xffffffffu, s_hh, o);
    }
    if (ph == 0) {
        a.part[((size_t)item * 2) * 32 + (pw & 31)] = s_dh;
        a.part[((size_t)item * 2 + 1) * 32 + (pw & 31)] = s_hh;
    }
}

// SMALL = 1 (batches of up to 1024 walkers; blocks of ONE warp): block b is group item b of the planner's table, as in
// k_full_fused<.., SMALL = 1>; one mode: lanes items too (fused_lanes_item_tf).
template <int NM1, int NC, bool WS, int SMALL = 0>
__global__ void __launch_bounds__(128, NC == 2 ? (NM1 ? (SMALL ? 4 : LL_TF_MINB) : 3) : 2) k_full_fused_tf(FusedArgs a)
{
    using TL = Tile<NC, WS>;
    constexpr int NCO = 8 + 8 * NC; // coefficients per (interval, mode)
    extern __shared__ __align__(128) double sm[];
    __shared__ __align__(8) uint64_t bar[2];
    __shared__ int s_lo, s_hi;

    const int tid = threadIdx.x;
    int p, tile, i0, i1, j_hint = 0;
    bool lanes_item = false;
    if (SMALL) {
        tile = blockIdx.x;
        if (tile >= __ldg(a.grp_tab + 32)) return;
        const int *it = a.grp_tab + grp_off_items() + tile;
        const int mi = gridDim.x; // the table's row length = the grid
        i0 = __ldg(it + mi);
        i1 = __ldg(it + 2 * mi);
        j_hint = __ldg(it + 3 * mi);
        const int code = __ldg(it);
        lanes_item = NM1 && LL_SMALL_LANES && code < 0;
        p = lanes_item ? (-code - 1) + tid % kLW : code * 32 + tid;
    } else {
        p = blockIdx.x * blockDim.x + tid;
        tile = blockIdx.y;
        i0 = __ldg(a.tile_start + tile);
        i1 = __ldg(a.tile_start + tile + 1); // tile = dense bins [i0, i1)
    }
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
    if (blo >= bhi) {
        if (SMALL) { a.part[((size_t)tile * 2) * 32 + tid] = 0.0; a.part[((size_t)tile * 2 + 1) * 32 + tid] = 0.0; } // F4 reads every item
        return;
    }

    if (SMALL && NM1 && LL_SMALL_LANES && lanes_item) {
        fused_lanes_item_tf<NC, WS>(a, p, lo, hi, blo, bhi, j_hint, tile, sm, bar);
        return;
    }
    const int CH = a.CH;
    const int c_begin = blo / CH, c_end = (bhi + CH - 1) / CH;
    if (tid == 0) TL::issue(a, sm, c_begin, CH, &bar[0]);

    const size_t sw = (size_t)a.n_wp;
    const size_t cm = (size_t)NCO * sw;         // one mode's block
    const size_t cj = (size_t)a.n_m * cm;       // one interval's block
    const int kbase = (int)a.k_min;
    int j = SMALL ? j_hint : find_interval_of_bin(a.bstart, a.n_nodes, blo);
    int jl = -1;
    double co[NCO];
    double nxj = 0.0, sh0 = 0.0, s_dh = 0.0, s_hh = 0.0;
    double ts4 = 0.0; // 4 t_shift (reading R32)
    if (a.t_shift) {
        const int w = a.perm[p];
        if (w >= 0) ts4 = 4.0 * a.t_shift[(size_t)w * a.ts_stride];
    }

    for (int c = c_begin; c < c_end; ++c) {
        const int st = (c - c_begin) & 1;
        const uint32_t ph = (uint32_t)((c - c_begin) >> 1) & 1u;
        if (tid == 0 && c + 1 < c_end) TL::issue(a, sm + (size_t)(st ^ 1) * CH * TL::DPB, c + 1, CH, &bar[st ^ 1]);
        mbar_wait(&bar[st], ph);
        const double *sg = sm + (size_t)st * CH * TL::DPB;
        const int cb = c * CH;
        const double *sgc = sg - (size_t)cb * 2 * NC;
        const double *sWc = sg + (size_t)CH * 2 * NC - cb;
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
                    const double xj = __ldg(a.xj + j);
                    nxj = -xj;
                    sh0 = a.t_shift ? qc_linear_mod_cycle(xj, ts4) : 0.0;
                    if (NM1) {
#pragma unroll
                        for (int q = 0; q < NCO; ++q) co[q] = cc0[(size_t)q * sw];
                        if (a.t_shift) { co[4] += sh0; co[5] += ts4; }
                    }
                    jl = j;
                }
                // h^c of one mode at offset t from the interval's node, added into h
                auto mode_at = [&](double t, double (&h)[2 * NC]) {
                    const double A = cubic4(co, t), y = cubic4(co + 4, t);
                    double tf[2 * NC];
#pragma unroll
                    for (int q = 0; q < 2 * NC; ++q) tf[q] = cubic4(co + 8 + 4 * q, t);
                    double u, v; // h_m = u - i v
                    amp_expi_qc(A, y, u, v);
                    apply_tf<NC>(tf, u, v, h);
                };
                auto direct_bins = [&](int b0, int b1) {
                    if constexpr (!NM1) {
                        // several modes: chunks of four bins, mode loop outside (the coefficients read once per chunk)
                        for (int c4 = b0; c4 < b1; c4 += 4) {
                            double t4[4], h4[4][2 * NC];
#pragma unroll
                            for (int k = 0; k < 4; ++k) {
                                t4[k] = fma((double)(kbase + c4 + k), a.df, nxj);
#pragma unroll
                                for (int q = 0; q < 2 * NC; ++q) h4[k][q] = 0.0;
                            }
#pragma unroll 1
                            for (int m = 0; m < a.n_m; ++m) {
                                const double *cc = cc0 + (size_t)m * cm;
#pragma unroll
                                for (int q = 0; q < NCO; ++q) co[q] = cc[(size_t)q * sw];
                                if (a.t_shift) { co[4] += sh0; co[5] += ts4; }
#pragma unroll
                                for (int k = 0; k < 4; ++k) mode_at(t4[k], h4[k]);
                            }
#pragma unroll
                            for (int k = 0; k < 4; ++k) {
                                const int ii = c4 + k;
                                if (ii < b1 && ii >= tlo && ii < thi) accumulate_bin<NC, WS>(sgc, sWc, CH, ii, h4[k], s_dh, s_hh);
                            }
                        }
                    } else {
#pragma unroll 2
                        for (int ii = b0; ii < b1; ++ii) {
                            const bool act = (ii >= tlo) && (ii < thi);
                            const double t = fma((double)(kbase + ii), a.df, nxj);
                            double h[2 * NC];
#pragma unroll
                            for (int q = 0; q < 2 * NC; ++q) h[q] = 0.0;
                            mode_at(t, h);
                            if (act) accumulate_bin<NC, WS>(sgc, sWc, CH, ii, h, s_dh, s_hh);
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
                    LL_ROT_SINCOS(6.0 * co[7] * df3, su, cu);
                    unit_modulus(cu, su);
                    for (int k0 = flo; k0 < fhi; k0 += kRotSync) {
                        const int k1 = min(k0 + kRotSync, fhi);
                        const double t0 = fma((double)(kbase + k0), df, nxj);
                        const double tt = fma(2.0, t0, df), q3 = fma(3.0 * t0, t0 + df, df2), t1 = t0 + df;
                        double A = cubic4(co, t0);
                        double d1A = df * fma(co[3], q3, fma(co[2], tt, co[1]));
                        double d2A = df2 * fma(6.0 * co[3], t1, 2.0 * co[2]);
                        double sz, cz, sw_, cw, sv, cv;
                        LL_ROT_SINCOS(cubic4(co + 4, t0), sz, cz);
                        LL_ROT_SINCOS(df * fma(co[7], q3, fma(co[6], tt, co[5])), sw_, cw);
                        LL_ROT_SINCOS(df2 * fma(6.0 * co[7], t1, 2.0 * co[6]), sv, cv);
                        unit_modulus(cz, sz); unit_modulus(cw, sw_); unit_modulus(cv, sv);
#pragma unroll 2
                        for (int ii = k0; ii < k1; ++ii) {
                            const double t = fma((double)(kbase + ii), df, nxj);
                            const double u = A * cz, v = A * sz; // h = u - i v
                            double h[2 * NC];
#pragma unroll
                            for (int cch = 0; cch < NC; ++cch) {
                                const double tr = cubic4(co + 8 + 8 * cch, t), ti = cubic4(co + 12 + 8 * cch, t);
                                h[2 * cch] = fma(tr, u, ti * v);
                                h[2 * cch + 1] = fma(ti, u, -(tr * v));
                            }
                            accumulate_bin<NC, WS>(sgc, sWc, CH, ii, h, s_dh, s_hh);
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
        poison_stage(sg, CH * TL::DPB);
        __syncthreads();
    }
    if (SMALL) {
        a.part[((size_t)tile * 2) * 32 + tid] = s_dh;
        a.part[((size_t)tile * 2 + 1) * 32 + tid] = s_hh;
        return;
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

// F2 with per-walker nodes for FEW systems (Module-1 sized batches): k_spline_pw above is one thread per system walking
// 2 (n - 2) dependent rows, each with a division and a parked value (measured 0.81 ms for 320 systems of 1024 nodes: 760 cycles
// per row).  Here a block takes NWK neighbouring walkers of one system, thread = (chunk thread, walker), as k_spline_block4:
//  (a) the elimination factors c'_j = c_j / (b_j - a_j c'_{j-1}): no scan needed — the map contracts by <= 1/12 per row for
//      ANY node spacing (a_j c_j / den_j^2 with den_j >= h_{j-1}/4 + h_j/3 >= 2 sqrt(h_{j-1} h_j / 12)), so a thread that
//      starts kPwWarm = 16 rows before its chunk from c' = 0 has its chunk's first factor to 12^-16 < 1e-17 (from row 1 on
//      exactly: the true start);
//  (b) dp_j = (r_j - a_j dp_{j-1}) / den_j and (c) M_j = dp_j - c'_j M_{j+1}: first-order linear recurrences, by the scans
//      of affine maps of k_spline_block4.
// Same rows (and not-a-knot substitutions) as k_spline_pw; results equal to rounding.  Shared memory: xs, ys, cps, ds [n][NWK].
constexpr int kPwWarm = 16;
template <int NWK>
__global__ void __launch_bounds__(1024)
k_spline_pw_block(const double *__restrict__ Y, const double *__restrict__ X, double *__restrict__ C, int n_wp, int n_nodes, int n_m,
                  int bc)
{
    extern __shared__ double ssm[];
    __shared__ double sA[128], sB[128];
    const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31, wid = tid >> 5, nwarp = T >> 5;
    const int wl = tid % NWK, ct = tid / NWK, TT = T / NWK;
    const int nq = n_wp / NWK;
    const int sys = blockIdx.x / nq, p0 = (blockIdx.x - sys * nq) * NWK;
    const int m = sys >> 1, kind = sys & 1;
    const int n = n_nodes;
    const size_t sw = (size_t)n_wp;
    double *xs = ssm, *ys = xs + NWK * n, *cps = ys + NWK * n, *ds = cps + NWK * n, *xch = ds + NWK * n;
    for (int idx = tid; idx < NWK * n; idx += T) {
        const int j = idx / NWK;
        xs[idx] = __ldg(X + (size_t)j * sw + p0 + wl);
        ys[idx] = __ldg(Y + ((size_t)sys * n + j) * sw + p0 + wl);
    }
    __syncthreads();
    auto xv = [&](int j) { return xs[NWK * j + wl]; };
    auto yv = [&](int j) { return ys[NWK * j + wl]; };
    // row j (1 <= j <= n - 2) of the walker's system: a, b, c and the right-hand side r
    auto row = [&](int j, double &a, double &b, double &c, double &r) {
        const double hm = xv(j) - xv(j - 1), hp = xv(j + 1) - xv(j);
        a = hm * kSixth; b = (hm + hp) * (1.0 / 3.0); c = hp * kSixth;
        if (bc) { // not-a-knot: end conditions substituted into rows 1 and n - 2
            if (j == 1) { const double rho0 = hm / hp; b += a * (1.0 + rho0); c -= a * rho0; }
            if (j == n - 2) { const double rhon = hp / hm; b += c * (1.0 + rhon); a -= c * rhon; c = 0.0; }
        }
        if (j == 1) a = 0.0;
        r = (yv(j + 1) - yv(j)) / hp - (yv(j) - yv(j - 1)) / hm;
    };
    const int L = (n + TT - 1) / TT;
    const int j0 = min(ct * L, n), j1 = min(j0 + L, n);
    // ---- (a) c'_j of the chunk, after a warm-up of kPwWarm rows; (b) composed with the chunk's map for dp
    double cp = 0.0;
    for (int j = max(1, j0 - kPwWarm); j < min(j0, n - 1); ++j) {
        double a, b, c, r;
        row(j, a, b, c, r);
        cp = c / (b - a * cp);
    }
    double A = 0.0, B = 1.0;
    for (int j = j0; j < j1; ++j) {
        if (j >= 1 && j <= n - 2) {
            double a, b, c, r;
            row(j, a, b, c, r);
            const double inv = 1.0 / (b - a * cp);
            cp = c * inv;
            cps[NWK * j + wl] = cp;
            const double be = -a * inv;
            A = fma(be, A, r * inv);
            B *= be;
        } else cps[NWK * j + wl] = 0.0;
    }
    affine_scan4_up<NWK>(A, B, sA, sB, lane, wid, nwarp, wl);
    xch[tid] = A;
    __syncthreads();
    double dp = ct ? xch[tid - NWK] : 0.0;
    for (int j = j0; j < j1; ++j) {
        if (j >= 1 && j <= n - 2) {
            double a, b, c, r;
            row(j, a, b, c, r);
            const double cpm = (j >= 2) ? cps[NWK * (j - 1) + wl] : 0.0;
            dp = (r - a * dp) / (b - a * cpm);
            ds[NWK * j + wl] = dp;
        } else ds[NWK * j + wl] = 0.0;
    }
    __syncthreads();
    // ---- (c) backward sweep: M_j = dp_j - c'_j M_{j+1}
    A = 0.0; B = 1.0;
    for (int j = j1 - 1; j >= j0; --j) {
        if (j >= 1 && j <= n - 2) {
            const double be = -cps[NWK * j + wl];
            A = fma(be, A, ds[NWK * j + wl]);
            B *= be;
        } else { A = 0.0; B = 0.0; }
    }
    affine_scan4_down<NWK>(A, B, sA, sB, lane, wid, nwarp, wl);
    xch[tid] = A;
    __syncthreads();
    double Mn = (ct + 1 < TT) ? xch[tid + NWK] : 0.0;
    for (int j = j1 - 1; j >= j0; --j) {
        Mn = (j >= 1 && j <= n - 2) ? fma(-cps[NWK * j + wl], Mn, ds[NWK * j + wl]) : 0.0;
        ds[NWK * j + wl] = Mn;
    }
    __syncthreads();
    if (bc) {
        if (ct == 0) {
            const double rho0 = (xv(1) - xv(0)) / (xv(2) - xv(1)), rhon = (xv(n - 1) - xv(n - 2)) / (xv(n - 2) - xv(n - 3));
            ds[wl] = (1.0 + rho0) * ds[NWK + wl] - rho0 * ds[2 * NWK + wl];
            ds[NWK * (n - 1) + wl] = (1.0 + rhon) * ds[NWK * (n - 2) + wl] - rhon * ds[NWK * (n - 3) + wl];
        }
        __syncthreads();
    }
    double *c = C + ((size_t)m * 8 + kind * 4) * sw + p0 + wl;
    const size_t cj = (size_t)n_m * 8 * sw;
    for (int idx = tid; idx < NWK * (n - 1); idx += T) {
        const int j = idx / NWK;
        const double y0 = ys[idx], y1 = ys[idx + NWK], Mj = ds[idx], Mn1 = ds[idx + NWK];
        const double h = xs[idx + NWK] - xs[idx], ih = 1.0 / h;
        double *cc = c + (size_t)j * cj;
        cc[0] = y0;
        cc[sw] = (y1 - y0) * ih - h * (2.0 * Mj + Mn1) * kSixth;
        cc[2 * sw] = 0.5 * Mj;
        cc[3 * sw] = (Mn1 - Mj) * ih * kSixth;
    }
}

// F3 with per-walker intervals.  Same mapping and data staging as k_full_fused_tf (one thread = one walker, TMA-fed
// g/W tiles broadcast from shared memory); every lane tracks its own interval: the bins go up, so the interval index
// only moves forward, by a comparison with the lane's next node per bin.  NM1: the 8 coefficients of the lane's
// current interval live in registers; otherwise they are re-read per bin through L1.
#ifndef LL_PW_MINB
#define LL_PW_MINB 3
#endif
// SMALL = 1: one-warp blocks over the planner's group items (cost = bins: no interval table is shared by the walkers).
template <int NM1, int NC, bool WS, int SMALL = 0>
__global__ void __launch_bounds__(128, NM1 ? LL_PW_MINB : 3) k_full_fused_pw(FusedArgs a, const double *__restrict__ X)
{
    using TL = Tile<NC, WS>;
    extern __shared__ __align__(128) double sm[];
    __shared__ __align__(8) uint64_t bar[2];
    __shared__ int s_lo, s_hi;

    const int tid = threadIdx.x;
    int p, tile, i0, i1;
    if (SMALL) {
        tile = blockIdx.x;
        if (tile >= __ldg(a.grp_tab + 32)) return;
        const int *it = a.grp_tab + grp_off_items() + tile;
        const int mi = gridDim.x;
        i0 = __ldg(it + mi);
        i1 = __ldg(it + 2 * mi);
        p = __ldg(it) * 32 + tid;
    } else {
        p = blockIdx.x * blockDim.x + tid;
        tile = blockIdx.y;
        i0 = __ldg(a.tile_start + tile);
        i1 = __ldg(a.tile_start + tile + 1);
    }
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
    if (blo >= bhi) {
        if (SMALL) { a.part[((size_t)tile * 2) * 32 + tid] = 0.0; a.part[((size_t)tile * 2 + 1) * 32 + tid] = 0.0; } // F4 reads every item
        return;
    }

    const int CH = a.CH;
    const int c_begin = blo / CH, c_end = (bhi + CH - 1) / CH;
    if (tid == 0) TL::issue(a, sm, c_begin, CH, &bar[0]);

    const size_t sw = (size_t)a.n_wp;
    const size_t cm = (size_t)8 * sw, cj = (size_t)a.n_m * cm;
    const int n = a.n_nodes;
    const double *x = X + p;
    double ts4 = 0.0; // 4 t_shift (reading R32), folded into the phase cubic of the lane's current interval
    if (a.t_shift) {
        const int w = a.perm[p];
        if (w >= 0) ts4 = 4.0 * a.t_shift[(size_t)w * a.ts_stride];
    }
    // this lane's interval at its first bin: largest j in [0, n-2] with x_j <= f
    int j = 0;
    double xj = 0.0, xnext = INFINITY, sh0 = 0.0;
    double co[8];
    auto load_interval = [&](int jj) {
        xj = __ldg(x + (size_t)jj * sw);
        xnext = (jj < n - 2) ? __ldg(x + (size_t)(jj + 1) * sw) : INFINITY;
        sh0 = a.t_shift ? qc_linear_mod_cycle(xj, ts4) : 0.0;
        if (NM1) {
            const double *cc = a.C + (size_t)jj * cj + p;
#pragma unroll
            for (int q = 0; q < 8; ++q) co[q] = cc[(size_t)q * sw];
            if (a.t_shift) { co[4] += sh0; co[5] += ts4; }
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
    double tf1[2 * NC]; // single mode: the walker's transfer factors stay in registers
#pragma unroll
    for (int q = 0; q < 2 * NC; ++q) tf1[q] = NM1 ? a.TF[(size_t)q * sw + p] : 0.0;
    double s_dh = 0.0, s_hh = 0.0;

    for (int c = c_begin; c < c_end; ++c) {
        const int st = (c - c_begin) & 1;
        const uint32_t ph = (uint32_t)((c - c_begin) >> 1) & 1u;
        if (tid == 0 && c + 1 < c_end) TL::issue(a, sm + (size_t)(st ^ 1) * CH * TL::DPB, c + 1, CH, &bar[st ^ 1]);
        mbar_wait(&bar[st], ph);
        const double *sg = sm + (size_t)st * CH * TL::DPB;
        const int cb = c * CH;
        const double *sgc = sg - (size_t)cb * 2 * NC;
        const double *sWc = sg + (size_t)CH * 2 * NC - cb;
        const int tlo = max(cb, lo), thi = min(cb + CH, hi);
        auto one_bin = [&](int ii, double f) {
            const double t = f - xj;
            double h[2 * NC];
#pragma unroll
            for (int q = 0; q < 2 * NC; ++q) h[q] = 0.0;
            const int n_m = NM1 ? 1 : a.n_m;
            for (int m = 0; m < n_m; ++m) {
                if (!NM1) {
                    const double *cc = a.C + (size_t)j * cj + (size_t)m * cm + p;
#pragma unroll
                    for (int q = 0; q < 8; ++q) co[q] = cc[(size_t)q * sw];
                    if (a.t_shift) { co[4] += sh0; co[5] += ts4; }
                    const double *tf = a.TF + (size_t)m * 2 * NC * sw + p;
#pragma unroll
                    for (int q = 0; q < 2 * NC; ++q) tf1[q] = tf[(size_t)q * sw];
                }
                const double A = cubic4(co, t), y = cubic4(co + 4, t);
                double u, v; // h_m = u - i v
                amp_expi_qc(A, y, u, v);
                apply_tf<NC>(tf1, u, v, h);
            }
            accumulate_bin<NC, WS>(sgc, sWc, CH, ii, h, s_dh, s_hh);
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
                LL_ROT_SINCOS(cubic4(co + 4, t), sz, cz);
                LL_ROT_SINCOS(df * fma(co[7], q3, fma(co[6], tt, co[5])), sw_, cw);
                LL_ROT_SINCOS(df2 * fma(6.0 * co[7], t1, 2.0 * co[6]), sv, cv);
                LL_ROT_SINCOS(6.0 * co[7] * df3, su, cu);
                unit_modulus(cz, sz); unit_modulus(cw, sw_); unit_modulus(cv, sv); unit_modulus(cu, su);
#pragma unroll 2
                for (int k = 0; k < m; ++k) {
                    const double u = A * cz, v = A * sz; // h = u - i v
                    double h[2 * NC];
#pragma unroll
                    for (int cch = 0; cch < NC; ++cch) {
                        h[2 * cch] = fma(tf1[2 * cch], u, tf1[2 * cch + 1] * v);
                        h[2 * cch + 1] = fma(tf1[2 * cch + 1], u, -(tf1[2 * cch] * v));
                    }
                    accumulate_bin<NC, WS>(sgc, sWc, CH, ii + k, h, s_dh, s_hh);
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
        poison_stage(sg, CH * TL::DPB);
        __syncthreads();
    }
    if (SMALL) {
        a.part[((size_t)tile * 2) * 32 + tid] = s_dh;
        a.part[((size_t)tile * 2 + 1) * 32 + tid] = s_hh;
        return;
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
// tile slices per block of the two F4 kernels: 32, or 16 when a walker has more than 5 partial sums (the slices meet in
// shared memory, [slices][NQ][32] doubles <= 48 KB)
__host__ __device__ constexpr int fin_slices(int nq) { return nq > 5 ? 16 : 32; }

template <int NQ>
__global__ void __launch_bounds__(32 * fin_slices(NQ))
k_reduce_tiles(const double *__restrict__ part, const int *__restrict__ ilo, const int *__restrict__ ihi, int n_wp,
               const int *__restrict__ tile_start, int n_tiles, int cs, double *__restrict__ part2)
{
    constexpr int FY = fin_slices(NQ);
    __shared__ double red[FY][NQ][32];
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
        for (int t = t0 + ty; t <= t1; t += FY) {
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
        for (int k = 1; k < FY; ++k) v += red[k][q][threadIdx.x];
        part2[((size_t)z * NQ + q) * sw + p] = v;
    }
}

// F4: reduce the per-tile partials in a fixed order, apply T^c (single mode), form log L        (Eq. 2)
// Block = 32 walkers x kFinY tile slices: slice ty sums tiles t0 + ty, t0 + ty + kFinY, ... of its walker, the
// slices meet in shared memory and are added in slice order (deterministic: reruns are bit-identical).
template <int NM1, int NC, int NW> // NW: weight rows behind the single-mode H sums (1 shared, NC per channel)
__global__ void __launch_bounds__(32 * fin_slices(NM1 ? 2 * NC + NW : 2))
k_finalize(const double *__restrict__ part, const double *__restrict__ TF, const int *__restrict__ perm,
           const int *__restrict__ ilo, const int *__restrict__ ihi, int n_wp, const int *__restrict__ tile_start,
           int n_tiles, const double *__restrict__ dd, double *__restrict__ logL, double *__restrict__ d_h,
           double *__restrict__ h_h)
{
    constexpr int NQ = NM1 ? 2 * NC + NW : 2;
    constexpr int kFinY = fin_slices(NQ);
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
        // Re sum_c T^c S^c,  sum_c |T^c|^2 H^c (one H for a shared weight row)
        dh = 0.0; hh = 0.0;
        double t2 = 0.0;
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const double tr = TF[(size_t)(2 * c) * sw + p], ti = TF[(size_t)(2 * c + 1) * sw + p];
            dh += tr * acc[2 * c] - ti * acc[2 * c + 1];
            if (NW == 1) t2 += tr * tr + ti * ti;
            else hh += (tr * tr + ti * ti) * acc[2 * NC + c];
        }
        if (NW == 1) hh = t2 * acc[2 * NC];
    } else {
        dh = acc[0];
        hh = acc[1];
    }
    logL[w] = dh - 0.5 * hh - 0.5 * dd[0];
    if (d_h) d_h[w] = dh;
    if (h_h) h_h[w] = hh;
}

// F4 for small batches (k_full_fused<.., SMALL = 1>).  A group's records are ~1000 x 1.3 KB, and ONE block pulling them
// through one SM took 19 us (ncu r02: 70 long-scoreboard stalls per issue), so a group is summed by kFinZ blocks: block z
// takes the items t = z (mod kFinZ) of every walker's range, its 32 slices every 32nd of those, in a fixed order; the
// block's sums go to part2[group][z], and the block that finishes last (a ticket per group) adds the kFinZ records in z
// order, applies T^c and forms log L — the same order whichever block comes last, so reruns are bit-identical.
constexpr int kFinZ = 8;
template <int NM1, int NC, int NW>
__global__ void __launch_bounds__(32 * fin_slices(NM1 ? 2 * NC + NW : 2))
k_finalize_small(const double *__restrict__ part, double *__restrict__ part2, const double *__restrict__ TF,
                 const int *__restrict__ perm, int n_wp, int *__restrict__ grp_tab, const double *__restrict__ dd,
                 double *__restrict__ logL, double *__restrict__ d_h, double *__restrict__ h_h)
{
    constexpr int NQ = NM1 ? 2 * NC + NW : 2;
    constexpr int FY = fin_slices(NQ);
    __shared__ double red[FY][NQ][32];
    __shared__ int s_last;
    const int grp = blockIdx.x, z = blockIdx.y, lane = threadIdx.x, ty = threadIdx.y;
    const int p = grp * 32 + lane;
    const size_t sw = (size_t)n_wp;
    double acc[NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) acc[q] = 0.0;
    // the group items the walker's band touches, then its own lanes items (its slot of their records)
#pragma unroll
    for (int range = 0; range < 2; ++range) {
        const int t0 = grp_tab[(range ? grp_off_tb0() : grp_off_t0()) + p], t1 = grp_tab[(range ? grp_off_tb1() : grp_off_t1()) + p];
        const int first = t0 + ((z - t0 % kFinZ) + kFinZ) % kFinZ; // the first of them with t = z (mod kFinZ)
#pragma unroll 4
        for (int t = first + ty * kFinZ; t <= t1; t += FY * kFinZ) {
            const double *o = part + (size_t)t * NQ * 32 + lane;
#pragma unroll
            for (int q = 0; q < NQ; ++q) acc[q] += o[q * 32];
        }
    }
#pragma unroll
    for (int q = 0; q < NQ; ++q) red[ty][q][lane] = acc[q];
    __syncthreads();
    double *rec = part2 + (size_t)grp * kFinZ * NQ * 32 + lane; // [z][NQ][32]
    if (ty == 0) {
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            double v = red[0][q][lane];
#pragma unroll
            for (int k = 1; k < FY; ++k) v += red[k][q][lane];
            rec[((size_t)z * NQ + q) * 32] = v;
        }
        __threadfence(); // the record is visible before the ticket is taken
    }
    __syncthreads();
    if (ty == 0 && lane == 0) s_last = atomicAdd(grp_tab + grp_off_ticket() + grp, 1) == kFinZ - 1;
    __syncthreads();
    if (!s_last || ty != 0) return;
    __threadfence();
    const int w = perm[p];
    if (w < 0) return;
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        double v = 0.0;
#pragma unroll
        for (int k = 0; k < kFinZ; ++k) v += __ldcg(rec + ((size_t)k * NQ + q) * 32); // L2: written by other SMs
        acc[q] = v;
    }
    double dh = 0.0, hh = 0.0;
    if (NM1) {
        double t2 = 0.0;
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const double tr = TF[(size_t)(2 * c) * sw + p], ti = TF[(size_t)(2 * c + 1) * sw + p];
            dh += tr * acc[2 * c] - ti * acc[2 * c + 1];
            if (NW == 1) t2 += tr * tr + ti * ti;
            else hh += (tr * tr + ti * ti) * acc[2 * NC + c];
        }
        if (NW == 1) hh = t2 * acc[2 * NC];
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
k_full_template(FusedArgs a, int p, int n_c, double *__restrict__ h_out)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.n_f) return;
    double h[2 * kMaxNC];
#pragma unroll
    for (int q = 0; q < 2 * kMaxNC; ++q) h[q] = 0.0;
    if (i >= a.ilo[p] && i < a.ihi[p]) {
        const int j = find_interval_of_bin(a.bstart, a.n_nodes, (int)i);
        const size_t sw = (size_t)a.n_wp;
        const double t = fma((double)(a.k_min + i), a.df, -a.xj[j]);
        double ysh = 0.0;
        if (a.t_shift && a.perm[p] >= 0) ysh = qc_linear_mod_cycle((double)(a.k_min + i) * a.df, 4.0 * a.t_shift[(size_t)a.perm[p] * a.ts_stride]);
        for (int m = 0; m < a.n_m; ++m) {
            const double *cc = a.C + ((size_t)j * a.n_m + m) * 8 * sw + p;
            const double A = fma(fma(fma(cc[3 * sw], t, cc[2 * sw]), t, cc[sw]), t, cc[0]);
            const double y = fma(fma(fma(cc[7 * sw], t, cc[6 * sw]), t, cc[5 * sw]), t, cc[4 * sw]) + ysh;
            double sn, cs;
            sincos_qc(y, sn, cs);
            const double u = A * cs, v = A * sn;
            const double *tf = a.TF + (size_t)m * 2 * n_c * sw + p;
#pragma unroll
            for (int c = 0; c < kMaxNC; ++c)
                if (c < n_c) {
                    const double tr = tf[(size_t)(2 * c) * sw], ti = tf[(size_t)(2 * c + 1) * sw];
                    h[2 * c] = fma(tr, u, h[2 * c]); h[2 * c] = fma(ti, v, h[2 * c]);
                    h[2 * c + 1] = fma(ti, u, h[2 * c + 1]); h[2 * c + 1] = fma(-tr, v, h[2 * c + 1]);
                }
        }
    }
#pragma unroll
    for (int c = 0; c < kMaxNC; ++c)
        if (c < n_c) reinterpret_cast<double2 *>(h_out)[(size_t)c * a.n_f + i] = make_double2(h[2 * c], h[2 * c + 1]);
}

// stand-in template of one parameter row evaluated directly at arbitrary frequencies (no spline, no tables)
struct DirectRow {
    double p[5 + 2 * kMaxNC * kMaxModes];
    double c_lm[kMaxModes];
};
struct DirectClm {
    double c_lm[kMaxModes];
};

// h^c (re, im per channel) of one stand-in parameter row at frequency fi, evaluated directly (Eq. 7, 9; reading R9)
__device__ __forceinline__ void direct_template_at(const double *__restrict__ rp, const double *__restrict__ c_lm,
                                                   const StandinInfo &si, double Mtot, double eta, double fisco,
                                                   double fi, double (&h)[2 * kMaxNC])
{
    const double tc = rp[2], phic = rp[3], invD = rp[4];
    const double inv_kappa = 1.0 / si.kappa;
#pragma unroll
    for (int q = 0; q < 2 * kMaxNC; ++q) h[q] = 0.0;
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
        const double *tf = rp + 5 + m * 2 * si.n_c;
#pragma unroll
        for (int c = 0; c < kMaxNC; ++c)
            if (c < si.n_c) {
                const double tr = tf[2 * c], ti = tf[2 * c + 1];
                h[2 * c] = fma(tr, u, h[2 * c]); h[2 * c] = fma(ti, vv, h[2 * c]);
                h[2 * c + 1] = fma(ti, u, h[2 * c + 1]); h[2 * c + 1] = fma(-tr, vv, h[2 * c + 1]);
            }
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
    double h[2 * kMaxNC];
#pragma unroll
    for (int q = 0; q < 2 * kMaxNC; ++q) h[q] = 0.0;
    if (fi >= f_lo && fi <= f_hi) {
        double Mtot, eta, fisco;
        standin_masses(row.p[0], row.p[1], Mtot, eta, fisco);
        direct_template_at(row.p, row.c_lm, si, Mtot, eta, fisco, fi, h);
    }
#pragma unroll
    for (int c = 0; c < kMaxNC; ++c)
        if (c < si.n_c) reinterpret_cast<double2 *>(h_out)[(size_t)c * n_freq + i] = make_double2(h[2 * c], h[2 * c + 1]);
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
template <int NC>
__global__ void __launch_bounds__(256)
k_het_audit(const double *__restrict__ params, int P, DirectClm cl, StandinInfo si, const double *__restrict__ g,
            const double *__restrict__ Wc, int w_rows, long long n_f_pad, GridInfo gi, const int *__restrict__ estart,
            int n_b, const double *__restrict__ dd, double *__restrict__ logL, double *__restrict__ d_h,
            double *__restrict__ h_h)
{
    __shared__ double sh[8];
    const size_t w = blockIdx.x;
    const double *rp = params + w * P;
    const int i_lo = estart[0], i_hi = estart[n_b];
    double Mtot, eta, fisco;
    standin_masses(rp[0], rp[1], Mtot, eta, fisco);
    double a_dh = 0.0, a_hh = 0.0;
    for (int i = i_lo + threadIdx.x; i < i_hi; i += blockDim.x) {
        double h[2 * kMaxNC];
        direct_template_at(rp, cl.c_lm, si, Mtot, eta, fisco, bin_freq(gi.k_min, i, gi.df), h);
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const double2 gg = reinterpret_cast<const double2 *>(g)[(size_t)i * NC + c]; // W conj(d)
            a_dh += gg.x * h[2 * c] - gg.y * h[2 * c + 1];
            a_hh = fma(Wc[(w_rows > 1 ? (size_t)c * n_f_pad : 0) + i], h[2 * c] * h[2 * c] + h[2 * c + 1] * h[2 * c + 1], a_hh);
        }
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
// raw[b][6 NC + 1]: per channel (A0r, A0i, A1r, A1i, B0, B1), then sum_c W^c |d^c|^2 over the bin.
// ---------------------------------------------------------------------------------------------------
template <int NC>
__global__ void __launch_bounds__(256)
k_het_prepare(const double *__restrict__ g, const double *__restrict__ Wc, int w_rows, long long n_f_pad,
              const double *__restrict__ h0, GridInfo gi, const int *__restrict__ estart, const double *__restrict__ fb,
              double *__restrict__ raw)
{
    constexpr int NR = 6 * NC + 1;
    __shared__ double sh[8];
    const int b = blockIdx.x;
    const int i_lo = estart[b], i_hi = estart[b + 1];
    const double f_b = fb[b];
    double acc[NR];
#pragma unroll
    for (int q = 0; q < NR; ++q) acc[q] = 0.0;
    for (int i = i_lo + threadIdx.x; i < i_hi; i += blockDim.x) {
        const double t = bin_freq(gi.k_min, i, gi.df) - f_b;
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            const double2 gg = reinterpret_cast<const double2 *>(g)[(size_t)i * NC + c]; // W conj(d): (W d_re, -W d_im)
            const double w = Wc[(w_rows > 1 ? (size_t)c * n_f_pad : 0) + i];
            const double2 hc = reinterpret_cast<const double2 *>(h0)[(size_t)c * gi.n_f + i];
            // W d conj(h0) = conj( (W conj d) h0 )
            const double pr = gg.x * hc.x - gg.y * hc.y, pi = -(gg.x * hc.y + gg.y * hc.x);
            const double q = w * (hc.x * hc.x + hc.y * hc.y);
            double *o = acc + 6 * c;
            o[0] += pr; o[1] += pi; o[2] = fma(pr, t, o[2]); o[3] = fma(pi, t, o[3]);
            o[4] += q; o[5] = fma(q, t, o[5]);
            // W |d|^2 = |W conj d|^2 / W
            if (w > 0.0) acc[6 * NC] += (gg.x * gg.x + gg.y * gg.y) / w;
        }
    }
#pragma unroll
    for (int q = 0; q < NR; ++q) {
        const double tot = block_sum_256(acc[q], sh);
        if (threadIdx.x == 0) raw[(size_t)b * NR + q] = tot;
    }
}

// ---------------------------------------------------------------------------------------------------
// H1-H3: heterodyned likelihood.  Packed table (host-built by ll_het_prepare), all in shared memory:
//   edge e : f4[e] = 4 f_e; ih0[e][2 NC] = 1/h0^c (re, im) per channel;
//            per mode m: cfp[m][e] = c_lm f_e^(-7/6), f2m[m][e] = 2 f_e/m, fm53[m][e] = (m/pi) (2 f_e/m)^(-5/3)
//   bin b  : [6 NC] = A0h[2 NC] = A0/2 (re, im per channel), A1w[2 NC] = A1/(e_{b+1}-e_b), B0q[NC] = B0/4,
//            B1w[NC] = B1/(e_{b+1}-e_b)
// With s = r_lo + r_hi and dlt = r_hi - r_lo:  r0 = s/2, r1 = dlt/width                         (Eq. 11), so
//   Z[d,h] term = Re[A0 conj r0 + A1 conj r1] = A0h . s + A1w . dlt                              (Eq. 14)
//   Z[h,h] term = B0 |r0|^2 + 2 B1 Re[r0 conj r1] = B0q |s|^2 + B1w (s . dlt)                    (Eq. 17)
// The per-channel weights (reading R5) enter only through the summary data, i.e. through ll_het_prepare.
// ---------------------------------------------------------------------------------------------------
struct HetTable {
    const double *base; // device copy of the packed table
    int n_e, n_b, n_m, n_c;
    int total;          // doubles
    __host__ __device__ int off_f4() const { return 0; }
    __host__ __device__ int off_ih0() const { return n_e; }
    __host__ __device__ int off_cfp() const { return (1 + 2 * n_c) * n_e; }
    __host__ __device__ int off_f2m() const { return (1 + 2 * n_c) * n_e + n_m * n_e; }
    __host__ __device__ int off_fm53() const { return (1 + 2 * n_c) * n_e + 2 * n_m * n_e; }
    __host__ __device__ int off_bins() const { return (1 + 2 * n_c) * n_e + 3 * n_m * n_e; }
    __host__ __device__ int bin_stride() const { return 6 * n_c; }
};

template <int NC>
__device__ __forceinline__ void het_bin_contract(const double *__restrict__ tb, const double (&l)[2 * NC],
                                                 const double (&h)[2 * NC], double &dh, double &hh)
{
    double s[2 * NC], d[2 * NC];
#pragma unroll
    for (int q = 0; q < 2 * NC; ++q) { s[q] = l[q] + h[q]; d[q] = h[q] - l[q]; }
#pragma unroll
    for (int q = 0; q < 2 * NC; ++q) dh = fma(tb[q], s[q], dh);
#pragma unroll
    for (int q = 0; q < 2 * NC; ++q) dh = fma(tb[2 * NC + q], d[q], dh);
#pragma unroll
    for (int c = 0; c < NC; ++c) hh = fma(tb[4 * NC + c], fma(s[2 * c], s[2 * c], s[2 * c + 1] * s[2 * c + 1]), hh);
#pragma unroll
    for (int c = 0; c < NC; ++c) hh = fma(tb[5 * NC + c], fma(s[2 * c], d[2 * c], s[2 * c + 1] * d[2 * c + 1]), hh);
}

// Stand-in parameters -> log L.  Block = 32 lanes x (G walker groups x S frequency segments) warps sharing ONE
// copy of the table: warp (g, s) walks segment s of the bins for the 32 walkers of group g.  Lanes of a warp
// are 32 different walkers at the same edge, so every table read is a broadcast.  Blocks stride over passes of
// G groups; the S partial sums of a group meet in shared memory in segment order (deterministic).
//
// Inside a segment the edges go in chunks of E = 4 with the MODE loop outside the edge loop: the transfer factors
// of a mode are read once per chunk (from a lane-major shared copy, so they do not occupy 2 NC n_m registers for
// the whole kernel), and the four edges of a chunk are four independent phase -> sincos -> T^c h chains in
// flight per thread (with 16 warps per SM the FP64 pipe needs that instruction-level parallelism).  Whether any
// lane needs the taper polynomial is decided once per chunk (warp-uniform), below f_ISCO m_min/2 it is 1.
struct HetEdgeCtx {
    const double *f4, *ih0, *cfp, *f2m, *fm53;
    const double *tfs; // shared: this lane's staged parameter row + 5, i.e. T^c_m (re, im) mode-major, [n_m][2 NC]
    const double *nmq; // shared, [n_m]: -(m/pi)
    int n_e;
    double tc, invD, inv_fisco, K, phi0, kappa, inv_kappa;
};

template <int NM, int NC, int E, bool TAPER>
__device__ __forceinline__ void het_eval_edges(const HetEdgeCtx &x, const StandinInfo &si, int e, double (&r)[E][2 * NC])
{
    double h[E][2 * NC], ftc[E];
#pragma unroll
    for (int k = 0; k < E; ++k) {
#pragma unroll
        for (int q = 0; q < 2 * NC; ++q) h[k][q] = 0.0;
        ftc[k] = x.f4[e + k] * x.tc;
    }
#pragma unroll 1
    for (int m = 0; m < NM; ++m) {
        const double nmq = x.nmq[m]; // -(m/pi), shared
        const double *tq = x.tfs + m * 2 * NC;
        double tf[2 * NC];
#pragma unroll
        for (int q = 0; q < 2 * NC; ++q) tf[q] = tq[q];
        const int t = m * x.n_e + e;
#pragma unroll
        for (int k = 0; k < E; ++k) {
            // quarter cycles: 4 f t_c + (m/pi) K (2f/m)^(-5/3) - (m/pi)(phi_c + pi/4)
            const double y = fma(x.K, x.fm53[t + k], fma(nmq, x.phi0, ftc[k]));
            double A = x.cfp[t + k] * x.invD;
            if (TAPER) A *= taper_nobranch(x.f2m[t + k] * x.inv_fisco, x.kappa, x.inv_kappa);
            double u, v; // h_m = u - i v
            amp_expi_qc(A, y, u, v);
            apply_tf<NC>(tf, u, v, h[k]);
        }
    }
#pragma unroll
    for (int k = 0; k < E; ++k) { // r = h * (1/h0)
        const double *g = x.ih0 + 2 * NC * (e + k);
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            r[k][2 * c] = h[k][2 * c] * g[2 * c] - h[k][2 * c + 1] * g[2 * c + 1];
            r[k][2 * c + 1] = h[k][2 * c] * g[2 * c + 1] + h[k][2 * c + 1] * g[2 * c];
        }
    }
}

#ifndef LL_HET_E
#define LL_HET_E 4   // edges per chunk (independent chains per thread)
#endif
#ifndef LL_HET_WY
#define LL_HET_WY 16 // warps per block (one block per SM: the table copy is shared by all of them)
#endif
template <int NM, int NC>
__global__ void __launch_bounds__(32 * LL_HET_WY)
k_het_standin(HetTable T, StandinInfo si, const double *__restrict__ params, int P, int n_w, int n_groups, int S,
              const double *__restrict__ dd, double *__restrict__ logL, double *__restrict__ d_h,
              double *__restrict__ h_h)
{
    constexpr int E = LL_HET_E;
    constexpr int BS = 6 * NC; // table doubles per bin
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
            // coalesced loads (instead of one warp reading 2 NC n_m strided values per lane while the others wait)
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
            double pr[1][2 * NC];
            if (__any_sync(0xffffffffu, x.f4[b0] * x_scale > 1.0)) het_eval_edges<NM, NC, 1, true>(x, si, b0, pr);
            else het_eval_edges<NM, NC, 1, false>(x, si, b0, pr);
            double prev[2 * NC];
#pragma unroll
            for (int q = 0; q < 2 * NC; ++q) prev[q] = pr[0][q];
            int e = b0 + 1;
            for (; e + E <= b1 + 1; e += E) {
                double r[E][2 * NC];
                if (__any_sync(0xffffffffu, x.f4[e + E - 1] * x_scale > 1.0)) het_eval_edges<NM, NC, E, true>(x, si, e, r);
                else het_eval_edges<NM, NC, E, false>(x, si, e, r);
#pragma unroll
                for (int k = 0; k < E; ++k) {
                    het_bin_contract<NC>(bins + BS * (e + k - 1), prev, r[k], dh, hh);
#pragma unroll
                    for (int q = 0; q < 2 * NC; ++q) prev[q] = r[k][q];
                }
            }
            for (; e <= b1; ++e) {
                double r[1][2 * NC];
                if (__any_sync(0xffffffffu, x.f4[e] * x_scale > 1.0)) het_eval_edges<NM, NC, 1, true>(x, si, e, r);
                else het_eval_edges<NM, NC, 1, false>(x, si, e, r);
                het_bin_contract<NC>(bins + BS * (e - 1), prev, r[0], dh, hh);
#pragma unroll
                for (int q = 0; q < 2 * NC; ++q) prev[q] = r[0][q];
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
// z_e = A(f_e) e^{-i Psi(f_e)} common to all channels, and Eq. 14 / Eq. 17 regroup exactly into sums over edges:
//   Z[d,h] = Re sum_c conj(T^c) sum_e conj(z_e) Q^c_e,
//            Q^c_e = conj(1/h0^c_e) (A0_{e-1}/2 + A1_{e-1}/D_{e-1} + A0_e/2 - A1_e/D_e)            (Eq. 11, 14)
//   Z[h,h] = sum_c |T^c|^2 ( sum_e |z_e|^2 P^c_e + sum_b Re[z_b conj(z_{b+1}) X^c_b] ),
//            P^c_e = |1/h0^c_e|^2 (B0_{e-1}/4 + B1_{e-1}/D_{e-1} + B0_e/4 - B1_e/D_e),
//            X^c_b = (B0_b/2) (1/h0^c_b) conj(1/h0^c_{b+1})                                         (Eq. 11, 17)
// (D_b = f_{b+1} - f_b; terms whose bin index falls outside [0, n_b) are absent; 2 Re[r0 conj r1] =
// (|r_hi|^2 - |r_lo|^2)/D.)  Same arithmetic as the bin-by-bin form up to rounding; 48 instead of 73 FP64 slots
// per (walker, bin) for two channels.  Table: 4 + 5 NC doubles per edge (f4, fm53, cfp, f2m, then Q^c (re, im) per
// channel, P^c per channel, X^c (re, im) per channel), resident in shared memory, every read a broadcast.
// ---------------------------------------------------------------------------------------------------
__host__ __device__ constexpr int het1_stride(int n_c) { return 4 + 5 * n_c; }

struct Het1Table {
    const double *base;
    int n_e, n_b;
};

// the sums of one walker over the edges [e0, e1) of the table (and the bins [e0, min(e1, n_b))): D^c = sum conj(z) Q^c
// (re, im), H^c = sum |z|^2 P^c + Re[z_b conj(z_{b+1}) X^c_b]; lanes of the warp are 32 walkers at the same edges
template <int NC>
__device__ __forceinline__ void het1_segment(const double *__restrict__ tab, int n_b, const StandinInfo &si,
                                             const WalkerConst &c, int e0, int e1, double (&D)[2 * NC], double (&H)[NC])
{
    constexpr int ST = het1_stride(NC);
    constexpr int oQ = 4, oP = 4 + 2 * NC, oX = 4 + 3 * NC; // offsets of Q, P, X inside an edge's row
    const double inv_kappa = 1.0 / si.kappa;
    const double mh_pi = (double)si.mode_m[0] / kPi;
    const double Kq = mh_pi * c.K, nphq = -mh_pi * (c.phi + 0.25 * kPi);
    auto edge = [&](const double *t, double &u, double &v, double &amp) {
        const double y = fma(t[0], c.tc, fma(Kq, t[1], nphq));
        amp = t[2] * c.invD * taper(t[3] * c.inv_fisco, si.kappa, inv_kappa);
        amp_expi_qc(amp, y, u, v); // z = u - i v
    };
    const double *t = tab + (size_t)e0 * ST;
    double up, vp, ap;
    edge(t, up, vp, ap);
    const int last = min(e1, n_b); // one past the last bin whose cross term this segment owns
    auto edge_terms = [&](const double *tt, double u, double v, double a) { // conj(z) Q and |z|^2 P of one edge
        const double a2 = a * a;
#pragma unroll
        for (int cc = 0; cc < NC; ++cc) {
            const double qr = tt[oQ + 2 * cc], qi = tt[oQ + 2 * cc + 1];
            D[2 * cc] = fma(u, qr, D[2 * cc]); D[2 * cc] = fma(-v, qi, D[2 * cc]);
            D[2 * cc + 1] = fma(u, qi, D[2 * cc + 1]); D[2 * cc + 1] = fma(v, qr, D[2 * cc + 1]);
            H[cc] = fma(a2, tt[oP + cc], H[cc]);
        }
    };
    auto cross_terms = [&](const double *tt, double u0, double v0, double u1, double v1) { // z_e conj(z_{e+1}) X
        const double wr = fma(u0, u1, v0 * v1), wi = fma(u0, v1, -(v0 * u1));
#pragma unroll
        for (int cc = 0; cc < NC; ++cc) {
            H[cc] = fma(wr, tt[oX + 2 * cc], H[cc]);
            H[cc] = fma(-wi, tt[oX + 2 * cc + 1], H[cc]);
        }
    };
    int e = e0;
    // chunks of kE bins: the kE next edges are kE independent phase -> sincos chains in flight per thread;
    // the taper polynomial is needed only where some lane is above its f_ISCO (one warp-uniform test per chunk)
    constexpr int kE = 4;
    for (; e + kE <= last; e += kE, t += kE * ST) {
        double un[kE], vn[kE], an[kE];
        const bool tapered = __any_sync(0xffffffffu, t[kE * ST + 3] * c.inv_fisco > 1.0);
#pragma unroll
        for (int k = 0; k < kE; ++k) {
            const double *tn = t + (k + 1) * ST;
            const double y = fma(tn[0], c.tc, fma(Kq, tn[1], nphq));
            double a = tn[2] * c.invD;
            if (tapered) a *= taper_nobranch(tn[3] * c.inv_fisco, si.kappa, inv_kappa);
            an[k] = a;
            amp_expi_qc(a, y, un[k], vn[k]);
        }
#pragma unroll
        for (int k = 0; k < kE; ++k) {
            const double *tt = t + k * ST;
            const double u0 = k ? un[k - 1] : up, v0 = k ? vn[k - 1] : vp, a0 = k ? an[k - 1] : ap;
            edge_terms(tt, u0, v0, a0);
            cross_terms(tt, u0, v0, un[k], vn[k]);
        }
        up = un[kE - 1]; vp = vn[kE - 1]; ap = an[kE - 1];
    }
    for (; e < e1; ++e, t += ST) {
        edge_terms(t, up, vp, ap);
        if (e < last) { // bin e = [e, e + 1]: needs z at e + 1 (the next segment's first edge at the boundary)
            double un, vn, an;
            edge(t + ST, un, vn, an);
            cross_terms(t, up, vp, un, vn);
            up = un; vp = vn; ap = an;
        }
    }
}

#ifndef LL_HET1_WY
#define LL_HET1_WY 16 // warps per block of the single-mode kernel (one block per SM shares the table copy)
#endif
#ifndef LL_HET1_MINB
#define LL_HET1_MINB 1
#endif
template <int NC>
__global__ void __launch_bounds__(32 * LL_HET1_WY, LL_HET1_MINB)
k_het_standin1(Het1Table T, StandinInfo si, const double *__restrict__ params, int P, int n_w, int n_groups, int S,
               const double *__restrict__ dd, double *__restrict__ logL, double *__restrict__ d_h,
               double *__restrict__ h_h)
{
    constexpr int ST = het1_stride(NC);
    constexpr int NR = 3 * NC;                               // partial sums per walker: D^c (re, im), H^c
    extern __shared__ __align__(16) double tab[];
    const int total = T.n_e * ST;
    double *red = tab + total + (total & 1); // [G][S][NR][32]
    for (int i = threadIdx.x + threadIdx.y * 32; i < total; i += 32 * blockDim.y) tab[i] = T.base[i];
    __syncthreads();
    const int G = blockDim.y / S, seg = threadIdx.y % S, gslot = threadIdx.y / S, lane = threadIdx.x;
    const int per = (T.n_e + S - 1) / S;
    const int e0 = seg * per, e1 = min(e0 + per, T.n_e); // this segment owns edges [e0, e1) and bins [e0, min(e1, n_b))
    const double ddb = dd[1];

    for (int base = blockIdx.x * G; base < n_groups; base += gridDim.x * G) {
        const int grp = base + gslot;
        const int w = grp * 32 + lane;
        const bool valid = grp < n_groups && w < n_w;
        const double *row = params + (size_t)(valid ? w : 0) * P;
        const WalkerConst c = standin_consts(row);
        double D[2 * NC], H[NC];
#pragma unroll
        for (int q = 0; q < 2 * NC; ++q) D[q] = 0.0;
#pragma unroll
        for (int q = 0; q < NC; ++q) H[q] = 0.0;
        if (grp < n_groups && e0 < e1) het1_segment<NC>(tab, T.n_b, si, c, e0, e1, D, H);
        if (S > 1) {
            double *rg = red + (size_t)gslot * S * (NR * 32);
            double *q = rg + seg * (NR * 32) + lane;
#pragma unroll
            for (int k = 0; k < 2 * NC; ++k) q[32 * k] = D[k];
#pragma unroll
            for (int k = 0; k < NC; ++k) q[32 * (2 * NC + k)] = H[k];
            __syncthreads();
            if (seg == 0) {
#pragma unroll
                for (int k = 0; k < 2 * NC; ++k) D[k] = 0.0;
#pragma unroll
                for (int k = 0; k < NC; ++k) H[k] = 0.0;
                for (int s = 0; s < S; ++s) {
                    const double *r = rg + s * (NR * 32) + lane;
#pragma unroll
                    for (int k = 0; k < 2 * NC; ++k) D[k] += r[32 * k];
#pragma unroll
                    for (int k = 0; k < NC; ++k) H[k] += r[32 * (2 * NC + k)];
                }
            }
        }
        if (seg == 0 && valid) {
            // Re sum_c conj(T^c) D^c,  sum_c |T^c|^2 H^c
            double dh = 0.0, hh = 0.0;
#pragma unroll
            for (int cc = 0; cc < NC; ++cc) {
                const double tr = row[5 + 2 * cc], ti = row[6 + 2 * cc];
                dh += tr * D[2 * cc] + ti * D[2 * cc + 1];
                hh += (tr * tr + ti * ti) * H[cc];
            }
            logL[w] = dh - 0.5 * hh - 0.5 * ddb;
            if (d_h) d_h[w] = dh;
            if (h_h) h_h[w] = hh;
        }
        if (S > 1) __syncthreads();
    }
}

// sin and cos of (x radians + lin quarter cycles): x is reduced by Cody-Waite, the small second term is added to the
// reduced argument (the linear phase term of reading R32 arrives already reduced modulo one cycle)
__device__ __forceinline__ void sincos_rad_plus_qc(double x, double lin, double &sn, double &cs)
{
    const double sh = __dadd_rn(x * kTwoOverPi, kMagic);
    const int q = __double2loint(sh);
    const double nd = __dadd_rn(sh, -kMagic);
    double r = fma(-nd, kPio2_1, x);
    r = fma(-nd, kPio2_2, r);
    r = fma(-nd, kPio2_3, r);
    sincos_qc(fma(r, kTwoOverPi, lin) + (double)(q & 3), sn, cs);
}

// Array entry point: amp_e, phase_e [n_w][n_m][n_e] (radians).  One warp per walker, lanes over edges (the
// arrays are walker-major, so this is the coalesced direction); neighbouring edges meet through a shuffle.
// t_shift [n_w] or nullptr: Psi_m(f_e) = phase_e + 2 pi f_e t_shift (reading R32).
template <int NC>
__global__ void __launch_bounds__(256)
k_het_arrays(HetTable T, const double *__restrict__ amp_e, const double *__restrict__ phase_e,
             const double *__restrict__ tf, const double *__restrict__ t_shift, int n_w, const double *__restrict__ dd,
             double *__restrict__ logL, double *__restrict__ d_h, double *__restrict__ h_h)
{
    constexpr int BS = 6 * NC;
    extern __shared__ __align__(16) double tab[];
    for (int i = threadIdx.x; i < T.total; i += blockDim.x) tab[i] = T.base[i];
    __syncthreads();
    const double *ih0 = tab + T.off_ih0(), *bins = tab + T.off_bins(), *f4 = tab + T.off_f4();
    const int lane = threadIdx.x & 31, wpb = blockDim.x >> 5;
    const double ddb = dd[1];
    for (int w = blockIdx.x * wpb + (threadIdx.x >> 5); w < n_w; w += gridDim.x * wpb) {
        double dh = 0.0, hh = 0.0;
        const double ts = t_shift ? t_shift[w] : 0.0;
        for (int base = 0; base < T.n_b; base += 31) {
            const int e = base + lane;
            double r[2 * NC];
#pragma unroll
            for (int q = 0; q < 2 * NC; ++q) r[q] = 0.0;
            if (e < T.n_e) {
                double h[2 * NC];
#pragma unroll
                for (int q = 0; q < 2 * NC; ++q) h[q] = 0.0;
                const double lin = t_shift ? qc_linear_mod_cycle(f4[e], ts) : 0.0; // 4 f_e t_shift quarter cycles
                for (int m = 0; m < T.n_m; ++m) {
                    const size_t idx = ((size_t)w * T.n_m + m) * T.n_e + e;
                    const double A = amp_e[idx];
                    double sn, cs;
                    if (t_shift) sincos_rad_plus_qc(phase_e[idx], lin, sn, cs);
                    else sincos_rad(phase_e[idx], sn, cs);
                    const double u = A * cs, v = A * sn;
                    const double *t4 = tf + ((size_t)w * T.n_m + m) * 2 * NC;
                    double tfr[2 * NC];
#pragma unroll
                    for (int q = 0; q < 2 * NC; ++q) tfr[q] = __ldg(t4 + q);
                    apply_tf<NC>(tfr, u, v, h);
                }
                const double *g = ih0 + 2 * NC * e;
#pragma unroll
                for (int c = 0; c < NC; ++c) {
                    r[2 * c] = h[2 * c] * g[2 * c] - h[2 * c + 1] * g[2 * c + 1];
                    r[2 * c + 1] = h[2 * c] * g[2 * c + 1] + h[2 * c + 1] * g[2 * c];
                }
            }
            double nx[2 * NC];
#pragma unroll
            for (int q = 0; q < 2 * NC; ++q) nx[q] = __shfl_down_sync(0xffffffffu, r[q], 1);
            if (lane < 31 && e < T.n_b) het_bin_contract<NC>(bins + BS * e, r, nx, dh, hh);
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

// ---------------------------------------------------------------------------------------------------
// The whole sampler loop on the heterodyned likelihood in ONE launch (4e8 heterodyned evaluations
// are the paper's whole cost, a Module-2 iteration is 4000 of them).  A cooperative grid of one block per SM keeps the
// single-mode summary table (k_het_standin1's Q, P, X form) in shared memory for all n_iter iterations and runs, per
// iteration: [uniforms -> propose -> H1-H3 -> accept] for half 0, grid barrier, the same for half 1, grid barrier,
// the temperature-swap sweep (one warp per walker column), grid barrier.  Uniforms are the counter-based ones of
// reading R31, computed where they are used (no buffer), every arithmetic step is the one of k_pt_propose /
// k_het_standin1 / k_pt_accept / k_pt_swap_warp, so a run is the same pure function of (seed, iter0, state).
// Block = 32 lanes x WY warps: lanes are 32 proposals, warp s takes edge segment s of the table (S = WY segments).
// ---------------------------------------------------------------------------------------------------
struct PtRunArgs {
    double *x, *logL, *d_h, *h_h;       // [n_t][n_w][P], [n_t][n_w] (d_h, h_h may be null): read AND written in the loop
    const double *betas, *lo, *hi, *dd; // [n_t], [P], [P], dd[1] = <d|d> over the band
    unsigned long long *n_acc;          // [n_t] or null
    unsigned long long seed;
    long long iter0, n_iter;
    int n_t, n_w, n_dim;
    double a;
};

__device__ __forceinline__ double pt_uniform(unsigned long long seed, long long it, int kind, long long index)
{
    const unsigned long long G = 0x9E3779B97F4A7C15ull;
    const unsigned long long k = splitmix_mix(seed + G * (unsigned long long)(8 * it + kind + 1));
    const unsigned long long r = splitmix_mix(k + G * (unsigned long long)(index + 1));
    return (double)(r >> 11) * 0x1.0p-53;
}

#ifndef LL_PT_WY
#define LL_PT_WY 8 // warps (= edge segments) per block of the one-launch sampler: a pass of 32 proposals is bound by the FP64
                   // issue rate of ONE SM, so more warps only add barrier and reduction cost (measured at Module-2 size,
                   // half update: 16 warps 5.2 us, 8 warps 4.8 us)
#endif
template <int NC>
__global__ void __launch_bounds__(32 * LL_PT_WY, 1)
k_pt_run_het1(Het1Table T, StandinInfo si, PtRunArgs a)
{
    constexpr int ST = het1_stride(NC);
    constexpr int NR = 3 * NC;
    constexpr int P = 5 + 2 * NC;
    constexpr int S = LL_PT_WY;
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    extern __shared__ __align__(16) double tab[];
    const int total = T.n_e * ST;
    double *red = tab + total + (total & 1); // [S][NR][32]
    double *wc_s = red + S * NR * 32;        // [7][32]: the walker constants of the pass's 32 proposals, ln u_accept, (d-1) ln z
    constexpr int kSwapSlab = 32 * P + 16;   // per warp: a column's rows [32][P] and the source rung of every rung (swap sweep)
    double *swp = wc_s + 7 * 32;             // [S][kSwapSlab]
    for (int i = threadIdx.x + threadIdx.y * 32; i < total; i += 32 * blockDim.y) tab[i] = T.base[i];
    __syncthreads();
    const int seg = threadIdx.y, lane = threadIdx.x;
    const int per = (T.n_e + S - 1) / S;
    const int e0 = seg * per, e1 = min(e0 + per, T.n_e);
    const double ddb = a.dd[1];
    const int n_t = a.n_t, n_w = a.n_w, nh = n_w / 2, n_half = n_t * nh;
    const int n_pass = (n_half + 31) / 32;
    // the loop state is rewritten between grid barriers: plain (coherent) loads only, never the read-only path
    double *x = a.x, *logL = a.logL;

#ifdef LL_PT_TIMING // build-time debugging aid: where an iteration's time goes, as seen by block 0
    long long tm[4] = {0, 0, 0, 0}, t_a = 0, t_b = 0;
    auto now = []() { long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; };
#define LL_PT_TICK(v) v = now()
#define LL_PT_ADD(k, d) tm[k] += (d)
#else
#define LL_PT_TICK(v)
#define LL_PT_ADD(k, d)
#endif
    for (long long it = a.iter0; it < a.iter0 + a.n_iter; ++it) {
        for (int half = 0; half < 2; ++half) {
            LL_PT_TICK(t_a);
            const int k0 = half == 0 ? 0 : nh, j0 = half == 0 ? nh : 0;
            for (int pass = blockIdx.x; pass < n_pass; pass += gridDim.x) {
                const int i = pass * 32 + lane;
                const bool valid = i < n_half;
                const int ii = valid ? i : 0;
                const int t = ii / nh, k = ii - t * nh;
                // ---- proposal (k_pt_propose) and the walker constants, ONCE per proposal, by the first warp (with 16
                // segment warps each redoing pow, cbrt and three divisions for its 8 edges, the constants were more
                // than half of the block's FP64 instructions); the others pick the five constants up from shared memory
                double y[P], z = 1.0, l_old = 0.0, beta_t = 0.0;
                bool in = true;
                const size_t wk = (size_t)t * n_w + k0 + k;
                WalkerConst c;
                if (seg == 0) {
                    l_old = logL[wk];      // for the acceptance test: loaded here, with the rows, not on its critical path
                    beta_t = a.betas[t];
                    const double tt = __dadd_rn(__dmul_rn(a.a - 1.0, pt_uniform(a.seed, it, 3 * half, ii)), 1.0);
                    z = __ddiv_rn(__dmul_rn(tt, tt), a.a);
                    int j = (int)(pt_uniform(a.seed, it, 3 * half + 1, ii) * (double)nh);
                    j = min(max(j, 0), nh - 1);
                    const double *xk = x + wk * P;
                    const double *xj = x + ((size_t)t * n_w + j0 + j) * P;
#pragma unroll
                    for (int q = 0; q < P; ++q) {
                        const double xkq = xk[q], xjq = xj[q], lq = a.lo[q], hq = a.hi[q];
                        const double v = __dadd_rn(xjq, __dmul_rn(z, __dadd_rn(xkq, -xjq)));
                        in = in & (v >= lq) & (v <= hq);
                        y[q] = v;
                    }
                    if (!in) {
#pragma unroll
                        for (int q = 0; q < P; ++q) y[q] = xk[q];
                    }
                    c = standin_consts(y);
                    wc_s[lane] = c.tc; wc_s[32 + lane] = c.invD; wc_s[64 + lane] = c.inv_fisco; wc_s[96 + lane] = c.K;
                    wc_s[128 + lane] = c.phi;
                } else if (seg == 1) {
                    // the two logarithms of the acceptance test depend on the uniforms only: the second warp has them
                    // ready in shared memory before the first one needs them
                    const double tt = __dadd_rn(__dmul_rn(a.a - 1.0, pt_uniform(a.seed, it, 3 * half, ii)), 1.0);
                    const double zz = __ddiv_rn(__dmul_rn(tt, tt), a.a);
                    wc_s[160 + lane] = log(pt_uniform(a.seed, it, 3 * half + 2, ii));
                    wc_s[192 + lane] = (double)(a.n_dim - 1) * log(zz);
                }
                __syncthreads();
                if (seg != 0) {
                    c.tc = wc_s[lane]; c.invD = wc_s[32 + lane]; c.inv_fisco = wc_s[64 + lane]; c.K = wc_s[96 + lane];
                    c.phi = wc_s[128 + lane];
                }
                // ---- H1-H3 on the proposal (k_het_standin1)
                double D[2 * NC], H[NC];
#pragma unroll
                for (int q = 0; q < 2 * NC; ++q) D[q] = 0.0;
#pragma unroll
                for (int q = 0; q < NC; ++q) H[q] = 0.0;
                if (e0 < e1) het1_segment<NC>(tab, T.n_b, si, c, e0, e1, D, H);
                double *qd = red + seg * (NR * 32) + lane;
#pragma unroll
                for (int q = 0; q < 2 * NC; ++q) qd[32 * q] = D[q];
#pragma unroll
                for (int q = 0; q < NC; ++q) qd[32 * (2 * NC + q)] = H[q];
                __syncthreads();
                if (seg == 0 && valid) {
#pragma unroll
                    for (int q = 0; q < 2 * NC; ++q) D[q] = 0.0;
#pragma unroll
                    for (int q = 0; q < NC; ++q) H[q] = 0.0;
                    for (int s = 0; s < S; ++s) {
                        const double *r = red + s * (NR * 32) + lane;
#pragma unroll
                        for (int q = 0; q < 2 * NC; ++q) D[q] += r[32 * q];
#pragma unroll
                        for (int q = 0; q < NC; ++q) H[q] += r[32 * (2 * NC + q)];
                    }
                    double dh = 0.0, hh = 0.0;
#pragma unroll
                    for (int cc = 0; cc < NC; ++cc) {
                        const double tr = y[5 + 2 * cc], ti = y[6 + 2 * cc];
                        dh += tr * D[2 * cc] + ti * D[2 * cc + 1];
                        hh += (tr * tr + ti * ti) * H[cc];
                    }
                    const double l_new = dh - 0.5 * hh - 0.5 * ddb;
                    // ---- accept (k_pt_accept)
                    bool acc = false;
                    if (in && l_new == l_new && fabs(l_new) != INFINITY) {
                        const double lnq = __dadd_rn(wc_s[192 + lane], __dmul_rn(beta_t, __dadd_rn(l_new, -l_old)));
                        acc = wc_s[160 + lane] < lnq;
                    }
                    if (acc) {
                        double *xo = x + wk * P;
#pragma unroll
                        for (int q = 0; q < P; ++q) xo[q] = y[q];
                        logL[wk] = l_new;
                        if (a.d_h) a.d_h[wk] = dh;
                        if (a.h_h) a.h_h[wk] = hh;
                        if (a.n_acc) atomicAdd(a.n_acc + t, 1ull); // integer: order-independent
                    }
                }
                __syncthreads(); // red is reused by the next pass
            }
            LL_PT_TICK(t_b);
            grid.sync(); // the other half reads what this one wrote
            LL_PT_ADD(0, t_b - t_a);
            LL_PT_ADD(1, now() - t_b);
        }
        if (n_t > 1) {
            LL_PT_TICK(t_a);
            // ---- temperature swaps (reading R27; same decisions as k_pt_swap_warp): one warp per walker column.
            // Going down from the hottest rung, the cold partner of step t is always the ORIGINAL rung t - 1 (nothing has
            // touched it yet) and the hot one is whatever has been carried down so far, so the sweep is a scalar
            // recurrence on (carried log L, its source rung) — two FP64 operations and a compare per rung — after
            // which every rung knows which original row it ends up with and only the rows that moved are copied.
            for (int col = blockIdx.x * S + seg; col < n_w; col += gridDim.x * S) {
                const bool has = lane < n_t;
                const size_t cidx = (size_t)(has ? lane : 0) * n_w + col;
                const double l = has ? logL[cidx] : 0.0;
                const double dh = (has && a.d_h) ? a.d_h[cidx] : 0.0, hh = (has && a.h_h) ? a.h_h[cidx] : 0.0;
                const double beta = has ? a.betas[lane] : 0.0;
                // every rung's row of this column, loaded with the log L values (one memory round trip for the whole sweep, not
                // a second one after the cascade) and parked in the warp's shared-memory slab: element e = rung * P + parameter
                double *rows = swp + seg * kSwapSlab;
                int *srcs = reinterpret_cast<int *>(rows + 32 * P);
                const int ne = n_t * P;
                double rv[P];
#pragma unroll
                for (int k = 0; k < P; ++k) {
                    const int e = lane + 32 * k, t = e / P;
                    rv[k] = (e < ne) ? x[((size_t)t * n_w + col) * P + (e - t * P)] : 0.0;
                }
                const double lnu = (lane >= 1 && has) ? log(pt_uniform(a.seed, it, 6, (long long)(lane - 1) * n_w + col)) : 0.0;
                const double db = __dadd_rn(beta, -__shfl_up_sync(0xffffffffu, beta, 1)); // beta_t - beta_{t-1}
                const double lprev = __shfl_up_sync(0xffffffffu, l, 1);                  // ln L of rung t - 1
                double carried = __shfl_sync(0xffffffffu, l, n_t - 1);
                int csrc = n_t - 1, my_src = lane;
                for (int t = n_t - 1; t >= 1; --t) {
                    const double lu = __shfl_sync(0xffffffffu, lnu, t), d = __shfl_sync(0xffffffffu, db, t);
                    const double lc = __shfl_sync(0xffffffffu, lprev, t);
                    const bool sw = lu < __dmul_rn(d, __dadd_rn(lc, -carried));
                    if (lane == t) my_src = sw ? t - 1 : csrc;
                    if (!sw) { carried = lc; csrc = t - 1; }
                }
                if (lane == 0) my_src = csrc;
                if (has) srcs[lane] = my_src;
#pragma unroll
                for (int k = 0; k < P; ++k)
                    if (lane + 32 * k < ne) rows[lane + 32 * k] = rv[k];
                __syncwarp();
                const double l_new = __shfl_sync(0xffffffffu, l, my_src & 31);
                const double dh_new = __shfl_sync(0xffffffffu, dh, my_src & 31), hh_new = __shfl_sync(0xffffffffu, hh, my_src & 31);
                // only the rows that moved are written (all of them were read before the cascade)
#pragma unroll
                for (int k = 0; k < P; ++k) {
                    const int e = lane + 32 * k;
                    if (e < ne) {
                        const int t = e / P, q = e - t * P, src = srcs[t];
                        if (src != t) x[((size_t)t * n_w + col) * P + q] = rows[src * P + q];
                    }
                }
                __syncwarp(); // the slab is reused by the warp's next column
                if (has && my_src != lane) {
                    logL[cidx] = l_new;
                    if (a.d_h) a.d_h[cidx] = dh_new;
                    if (a.h_h) a.h_h[cidx] = hh_new;
                }
            }
            LL_PT_TICK(t_b);
            grid.sync();
            LL_PT_ADD(2, t_b - t_a);
            LL_PT_ADD(3, now() - t_b);
        }
    }
#ifdef LL_PT_TIMING
    if (blockIdx.x == 0 && threadIdx.x == 0 && threadIdx.y == 0)
        printf("pt_run phases per iteration (ns): half %.0f  sync %.0f  swap %.0f  sync %.0f\n", (double)tm[0] / (2.0 * a.n_iter),
               (double)tm[1] / (2.0 * a.n_iter), (double)tm[2] / a.n_iter, (double)tm[3] / a.n_iter);
#endif
#undef LL_PT_TICK
#undef LL_PT_ADD
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
