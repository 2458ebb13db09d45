// ll_b200.cu — host side of libll_b200.so: the C ABI of include/ll.h, workspace management, per-node-set and
// per-reference host tables, launch shapes.  All arithmetic of the method on the batch path runs in the
// kernels of ll_kernels.cuh; the host only builds walker-independent tables (Thomas factorisation of the
// shared-node spline matrix, bin->interval offsets, f^(-7/6) / f^(-5/3) node tables, 1/h0 at the edges).
//
// Build: nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -lineinfo -shared -Xcompiler -fPIC
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "ll.h"
#include "ll_kernels.cuh"

using namespace ll;

// Scratch of the one allocation-free entry point, ll_pt_stretch_half_het_static (include/ll.h): a file-scope device
// array of LL_STATIC_SCRATCH_BYTES that every GPU which loads this library holds until the process exits.  In host
// code this name is only the runtime's handle for the symbol, NOT a device address: the address a kernel may be given
// comes from cudaGetSymbolAddress (static_scratch_addr below), looked up once per device with that device current.
static __device__ __align__(256) double g_ll_static_scratch[LL_STATIC_SCRATCH_BYTES / sizeof(double)];

namespace {

// Every internal device buffer carries a guard band behind its capacity, filled with a canary byte when the block is
// allocated; ll_debug_check() reads the bands back and reports the buffers whose band was written (an out-of-bounds
// store by a kernel).  compute-sanitizer is closed on this pool, so this and the poisoned-stage build (LL_POISON_STAGES,
// ll_kernels.cuh) are the memory checks the tests run.
constexpr size_t kGuardBytes = 256;
constexpr int kGuardByte = 0xA5;
struct DevBuf {
    void *p = nullptr;
    size_t cap = 0;
    cudaError_t alloc(size_t bytes)
    {
        cudaError_t e = cudaMalloc(&p, bytes + kGuardBytes);
        if (e != cudaSuccess) { p = nullptr; return e; }
        cap = bytes;
        return cudaMemset((char *)p + cap, kGuardByte, kGuardBytes); // legacy stream: ordered before any later kernel
    }
    cudaError_t ensure(size_t bytes)
    {
        if (bytes <= cap) return cudaSuccess;
        if (p) {
            cudaError_t e = cudaFree(p); // synchronises the device: no kernel can still be using the old block
            p = nullptr;
            cap = 0;
            if (e != cudaSuccess) return e;
        }
        const size_t want = (bytes + bytes / 8 + 255) & ~(size_t)255;
        if (alloc(want) == cudaSuccess) return cudaSuccess;
        (void)cudaGetLastError();
        return alloc((bytes + 255) & ~(size_t)255);
    }
    // 0: guard band intact (or nothing allocated), 1: written, -1: the read-back failed
    int guard_state() const
    {
        if (!p) return 0;
        unsigned char h[kGuardBytes];
        if (cudaMemcpy(h, (const char *)p + cap, kGuardBytes, cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
        for (size_t i = 0; i < kGuardBytes; ++i)
            if (h[i] != kGuardByte) return 1;
        return 0;
    }
    void release()
    {
        if (p) cudaFree(p);
        p = nullptr;
        cap = 0;
    }
    template <typename T> T *as() const { return reinterpret_cast<T *>(p); }
};

struct FullPlan {
    int WB, TB, CH, n_tiles, n_wp, key_gran, n_keys;
};

} // namespace

struct ll_ctx {
    int device = 0, n_c = 2, n_m = 1, precision = 0, spline_bc = 0;
    int w_rows = 1; // weight rows kept on the device: 1 (two channels sharing their PSD) or n_c
    int sm_count = 148;
    std::string err;
    int64_t launches = 0;

    // F0 state
    bool have_data = false;
    long long n_f = 0, n_f_pad = 0, k_min = 0;
    double df = 0.0;
    DevBuf g, Wc, dd_part, dd;  // g [n_f_pad][2 n_c], Wc [w_rows][n_f_pad]; dd: [0] full grid, [1] het band
    DevBuf g4f, Wf, scale, wmax; // FP32-accumulate variant: g/sigma in binary32, W/sigma^2 in FP64, (sigma, 1/sigma, 1/sigma^2)
    DevBuf pairs;               // unsigned long long [1]

    // stand-in
    bool have_standin = false;
    StandinInfo si{};
    double c_lm[kMaxModes] = {0};
    int mode_l[kMaxModes] = {0};

    // node-set cache
    std::vector<double> nodes_host;
    bool nodes_valid = false;
    std::vector<int> bstart_host;  // bin -> interval table of the current node set (host copy)
    long long nodes_version = 0;   // bumped whenever the node tables are rebuilt
    // frequency-tile boundaries of the fused kernels [n_tiles + 1] (+ the chunk boundaries of the two-stage finalize):
    // one cached table per kind (0: uniform tiles, 1: small batches, tiles limited by the spline intervals they cross,
    // 2: per-walker node grids, uniform), keyed by (data version, node-set version, TB)
    struct TileCache {
        DevBuf tab;
        long long data_version = -1, nodes_version = -1;
        int TB = -1, n = 0, off2 = 0, n2 = 0;
    } tiles[3];
    TileCache *tile_cur = nullptr; // the table of the call in progress
    long long data_version = 0;    // bumped by every ll_set_data
    DevBuf part2;                  // chunk partials of the two-stage finalize
    DevBuf grp_tab;                // small batches: work items per group of 32 walkers (k_band_sort_small)
    DevBuf pw_x;                   // per-walker node grids: X [n_nodes][n_wp], then the effective bands [n_w][2]
    DevBuf node_tab; // doubles then ints
    DevBuf wmom;     // [w_rows][7][n_f_pad] prefix moments of every weight row inside the intervals of the current node set
    NodeTables nt{};

    // full-grid scratch
    DevBuf ilo_w, ihi_w, key_w, hist, perm, ilo_s, ihi_s, Y, C, TF, part, prow;
    int last_n_blocks = 0;

    // het state
    bool have_het = false;
    int n_e = 0;
    DevBuf het_tab, het_raw, het_idx, het_fb, het_tab1;
    DevBuf pt_u;                // ll_pt_run_*: the uniforms of one iteration
    DevBuf pt_y, pt_out, pt_in; // sampler step: proposals [n][P], (log L, <d|h>, <h|h>, (d-1) ln z) [4][n], inside flags
    DevBuf ref_idx, ref_dense, ref_edges; // ll_het_refresh_standin: argmax slot, h0 on the grid, h0 and f at the edges
    // launch shapes of the heterodyne kernels, per context (the shared-memory opt-in is per device, the
    // grid depends on this device's SM count)
    bool het1_attr = false, hetn_attr = false, heta_attr = false;
    size_t het1_bps_smem = 0;
    int het1_bps = 0;
    long long hetn_key_groups = -1;
    int hetn_key_total = -1, hetn_S = 1, hetn_grid = 1;
    bool pt_fused = true;          // ll_pt_run_het: the one-launch cooperative kernel when the population fits it
    int coop = -1;                 // device supports cooperative launches (-1: not asked yet)
    bool ptrun_attr = false;
    bool spl4_attr = false;
    bool hm_attr = false;
    bool splpw_attr = false;
    double *static_scratch = nullptr; // device address of g_ll_static_scratch on this context's device (ll_create)
    HetTable ht{};
    Het1Table ht1{}; // single-mode regrouped table (k_het_standin1); base == nullptr when not built
    std::vector<double> raw_host; // [n_b][6 n_c + 1]

    // host staging for the *_host entry points
    DevBuf stage_in, stage_out;

    // optional event bracketing of the dominant kernel (ll_profile_enable)
    bool profiling = false;
    std::vector<cudaEvent_t> ev; // pairs
    int ev_used = 0;             // pairs recorded since enable (ring)

    std::vector<std::pair<const char *, DevBuf *>> buffers()
    {
#define LL_B(x) {#x, &x}
        return {LL_B(g), LL_B(Wc), LL_B(dd_part), LL_B(dd), LL_B(pairs), LL_B(node_tab), LL_B(ilo_w), LL_B(ihi_w), LL_B(key_w),
                LL_B(hist), LL_B(perm), LL_B(ilo_s), LL_B(ihi_s), LL_B(Y), LL_B(C), LL_B(TF), LL_B(part), LL_B(prow),
                LL_B(het_tab), LL_B(het_tab1), LL_B(het_raw), LL_B(het_idx), LL_B(het_fb), LL_B(stage_in), LL_B(stage_out),
                LL_B(g4f), LL_B(Wf), LL_B(scale), LL_B(wmax), LL_B(ref_idx), LL_B(ref_dense), LL_B(ref_edges),
                LL_B(tiles[0].tab), LL_B(tiles[1].tab), LL_B(tiles[2].tab), LL_B(grp_tab), LL_B(wmom), LL_B(part2), LL_B(pw_x), LL_B(pt_y),
                LL_B(pt_out), LL_B(pt_in), LL_B(pt_u)};
#undef LL_B
    }
    int fail(int code, const std::string &msg)
    {
        err = msg;
        return code;
    }
    int cuda_fail(const char *what, cudaError_t e)
    {
        err = std::string(what) + ": " + cudaGetErrorString(e);
        (void)cudaGetLastError();
        return (e == cudaErrorMemoryAllocation) ? LL_ERR_NOMEM : LL_ERR_CUDA;
    }
};

namespace {

struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        if (prev != dev) cudaSetDevice(dev);
        else prev = -1;
    }
    ~DeviceGuard()
    {
        if (prev >= 0) cudaSetDevice(prev);
    }
};

#define CK(call)                                                           \
    do {                                                                   \
        cudaError_t e_ = (call);                                           \
        if (e_ != cudaSuccess) return ctx->cuda_fail(#call, e_);           \
    } while (0)

// device address of g_ll_static_scratch on `device`: one cudaGetSymbolAddress per device and process, made with that
// device current (a static __device__ array exists once per device, each copy at its own address)
constexpr int kMaxScratchDevices = 64;
std::mutex g_scratch_mu;
double *g_scratch_addr[kMaxScratchDevices] = {};
cudaError_t static_scratch_addr(int device, double **out)
{
    *out = nullptr;
    if (device < 0 || device >= kMaxScratchDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_scratch_mu);
    if (!g_scratch_addr[device]) {
        DeviceGuard dg(device);
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_ll_static_scratch);
        if (e != cudaSuccess) return e;
        g_scratch_addr[device] = static_cast<double *>(p);
    }
    *out = g_scratch_addr[device];
    return cudaSuccess;
}

#define LAUNCHED(ctx)                                                      \
    do {                                                                   \
        ++(ctx)->launches;                                                 \
        cudaError_t e_ = cudaGetLastError();                               \
        if (e_ != cudaSuccess) return (ctx)->cuda_fail("kernel launch", e_); \
    } while (0)

constexpr int kEvPairs = 512;

struct ProfScope { // records an event pair around one launch when profiling is on
    ll_ctx *ctx;
    cudaStream_t st;
    int slot = -1;
    ProfScope(ll_ctx *c, cudaStream_t s) : ctx(c), st(s)
    {
        if (ctx->profiling && !ctx->ev.empty()) {
            slot = ctx->ev_used % kEvPairs;
            cudaEventRecord(ctx->ev[2 * slot], st);
        }
    }
    ~ProfScope()
    {
        if (slot >= 0) {
            cudaEventRecord(ctx->ev[2 * slot + 1], st);
            ++ctx->ev_used;
        }
    }
};

inline int ceil_div(long long a, long long b) { return (int)((a + b - 1) / b); }

// the three data layouts the kernels are built for: (channels, one weight row shared by all of them?)
#define LL_LAYOUT(ctx, CALL)                                      \
    do {                                                          \
        if ((ctx)->n_c == 2 && (ctx)->w_rows == 1) { CALL(2, true); } \
        else if ((ctx)->n_c == 2) { CALL(2, false); }             \
        else { CALL(3, false); }                                  \
    } while (0)
#define LL_CHANNELS(ctx, CALL)                                    \
    do {                                                          \
        if ((ctx)->n_c == 2) { CALL(2); } else { CALL(3); }       \
    } while (0)
inline long long round_up(long long a, long long b) { return (a + b - 1) / b * b; }

// ---------------------------------------------------------------------------------------------------
// Node set: everything that depends on f_nodes and the dense grid only (cached across calls)
// ---------------------------------------------------------------------------------------------------
int prepare_nodes(ll_ctx *ctx, int n, const double *x, cudaStream_t st)
{
    if (ctx->nodes_valid && (int)ctx->nodes_host.size() == n && memcmp(ctx->nodes_host.data(), x, sizeof(double) * n) == 0)
        return LL_OK;
    ctx->nodes_valid = false;
    if (n < 3) return ctx->fail(LL_ERR_ARG, "n_nodes must be >= 3");
    if (n < 4 && ctx->spline_bc == LL_BC_NOT_A_KNOT) return ctx->fail(LL_ERR_ARG, "the not-a-knot boundary condition needs n_nodes >= 4");
    for (int j = 0; j + 1 < n; ++j)
        if (!(x[j + 1] > x[j])) return ctx->fail(LL_ERR_ARG, "f_nodes must be strictly ascending and finite");
    const double f_first = bin_freq(ctx->k_min, 0, ctx->df), f_last = bin_freq(ctx->k_min, ctx->n_f - 1, ctx->df);
    if (!(x[0] <= f_first) || !(x[n - 1] >= f_last))
        return ctx->fail(LL_ERR_ARG, "f_nodes do not cover the dense grid");
    if (!(x[0] > 0.0) && ctx->have_standin) return ctx->fail(LL_ERR_ARG, "f_nodes must be positive");

    const int n_m = ctx->n_m;
    const size_t nd = (size_t)n * (7 + 3 * (size_t)n_m); // doubles (hj/invh padded to n)
    std::vector<double> hd(nd, 0.0);
    std::vector<int> hi(n, 0);
    double *xj = hd.data(), *hj = xj + n, *invh = hj + n, *ta = invh + n, *tcp = ta + n, *tinv = tcp + n, *f4 = tinv + n;
    double *cfp = f4 + n, *f2m = cfp + (size_t)n_m * n, *fm53 = f2m + (size_t)n_m * n;
    typedef long double ld;
    for (int j = 0; j < n; ++j) {
        xj[j] = x[j];
        f4[j] = 4.0 * x[j];
    }
    for (int j = 0; j + 1 < n; ++j) {
        const ld h = (ld)x[j + 1] - (ld)x[j];
        hj[j] = (double)h;
        invh[j] = (double)(1.0L / h);
    }
    // Thomas factorisation of rows 1..n-2 of the spline system.  Natural: M_0 = M_{n-1} = 0.  Not-a-knot: the end
    // conditions M_0 = (1 + rho0) M_1 - rho0 M_2, M_{n-1} = (1 + rhon) M_{n-2} - rhon M_{n-3} (third derivative
    // continuous across x_1 and x_{n-2}) substituted into rows 1 and n-2, which stay tridiagonal.
    ld rho0 = 0.0L, rhon = 0.0L;
    if (ctx->spline_bc == LL_BC_NOT_A_KNOT) {
        rho0 = ((ld)x[1] - (ld)x[0]) / ((ld)x[2] - (ld)x[1]);
        rhon = ((ld)x[n - 1] - (ld)x[n - 2]) / ((ld)x[n - 2] - (ld)x[n - 3]);
    }
    {
        ld cprev = 0.0L;
        for (int j = 1; j <= n - 2; ++j) {
            const ld hm = (ld)x[j] - (ld)x[j - 1], hp = (ld)x[j + 1] - (ld)x[j];
            ld a = hm / 6.0L, b = (hm + hp) / 3.0L, c = hp / 6.0L;
            if (ctx->spline_bc == LL_BC_NOT_A_KNOT) {
                if (j == 1)     { b += a * (1.0L + rho0); c -= a * rho0; }
                if (j == n - 2) { b += c * (1.0L + rhon); a -= c * rhon; c = 0.0L; }
            }
            const ld den = (j == 1) ? b : b - a * cprev;
            const ld cp = c / den;
            ta[j] = (j == 1) ? 0.0 : (double)a;
            tcp[j] = (double)cp;
            tinv[j] = (double)(1.0L / den);
            cprev = cp;
        }
    }
    if (ctx->have_standin)
        for (int m = 0; m < n_m; ++m) {
            const ld mm = (ld)ctx->si.mode_m[m];
            for (int j = 0; j < n; ++j) {
                const ld f = (ld)x[j], fp = 2.0L * f / mm;
                cfp[(size_t)m * n + j] = (double)((ld)ctx->c_lm[m] * powl(f, -7.0L / 6.0L));
                f2m[(size_t)m * n + j] = (double)fp;
                fm53[(size_t)m * n + j] = (double)powl(fp, -5.0L / 3.0L);
            }
        }
    // bstart[j]: interval j covers dense bins [bstart[j], bstart[j+1]); lookup = largest j with x_j <= f,
    // clamped to [0, n-2] (reading R21)
    hi[0] = 0;
    for (int j = 1; j <= n - 2; ++j) hi[j] = (int)first_bin_ge(x[j], ctx->k_min, ctx->n_f, ctx->df);
    hi[n - 1] = (int)ctx->n_f;
    for (int j = 1; j < n; ++j) hi[j] = std::max(hi[j], hi[j - 1]);

    const size_t bytes_d = nd * sizeof(double), bytes_i = (size_t)n * sizeof(int);
    CK(ctx->node_tab.ensure(bytes_d + bytes_i));
    CK(cudaMemcpyAsync(ctx->node_tab.p, hd.data(), bytes_d, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync((char *)ctx->node_tab.p + bytes_d, hi.data(), bytes_i, cudaMemcpyHostToDevice, st));
    CK(cudaStreamSynchronize(st)); // the host vectors above go out of scope
    const double *b = ctx->node_tab.as<double>();
    NodeTables &nt = ctx->nt;
    nt.xj = b; nt.hj = b + n; nt.invh = b + 2 * n; nt.ta = b + 3 * n; nt.tcp = b + 4 * n; nt.tinv = b + 5 * n;
    nt.f4 = b + 6 * n; nt.cfp = b + 7 * n; nt.f2m = nt.cfp + (size_t)n_m * n; nt.fm53 = nt.f2m + (size_t)n_m * n;
    nt.bc = ctx->spline_bc; nt.rho0 = (double)rho0; nt.rhon = (double)rhon;
    nt.bstart = reinterpret_cast<const int *>((const char *)ctx->node_tab.p + bytes_d);
    ctx->nodes_host.assign(x, x + n);
    ctx->bstart_host = hi;
    ctx->nodes_version += 1;
    if (ctx->n_m == 1 && ctx->precision == LL_PREC_FP64) { // <h|h> by weight moments (single-mode kernel): one set per weight row
        CK(ctx->wmom.ensure(sizeof(double) * 7 * (size_t)ctx->w_rows * (size_t)ctx->n_f_pad));
        k_w_moments<<<dim3(n - 1, ctx->w_rows), 256, 0, st>>>(ctx->Wc.as<double>(), nt.bstart, nt.xj, n, ctx->k_min, ctx->df,
                                                              ctx->n_f_pad, ctx->wmom.as<double>());
        LAUNCHED(ctx);
    }
    ctx->nodes_valid = true;
    return LL_OK;
}

#ifndef LL_FUSED_CH
#define LL_FUSED_CH 512 // bins per TMA stage of the fused kernels (two stages per block): a block-wide barrier per stage;
                        // 256 -> 512 bins: 9.17 -> 9.08 ms at config 2 (40 KB per block, five blocks per SM)
#endif
FullPlan make_plan(const ll_ctx *ctx, long long n_w, bool hm_kernel = false) // hm_kernel: the launch may take k_full_fused_hm
{
    FullPlan pl;
    // blocks of 128 walkers above 1024 walkers (64-walker blocks between 1024 and 4096, as in round 1, measured worse: 2048
    // walkers on the config-2 grid frac 0.60 with 64 x 512-bin stages, 0.69 with 64 x 256, 0.73 with 128 x 512; 3072: 0.63 / 0.73 / 0.76)
    pl.WB = (n_w > 1024) ? 128 : (n_w >= 1024 ? 64 : 32);
    // three or six modes, the BASELINE layout, FP64 (k_full_fused_hm on both routes): the large route takes over a little below
    // 1024 walkers (six modes on the one-year grid, kernel on the small / large route: 320 walkers 2.71 / 4.01 ms, 512: 4.30 / 4.87,
    // 800: 6.71 / 8.63, 1024: 9.71 / 8.89)
    if (hm_kernel && (ctx->n_m == 3 || ctx->n_m == 6) && ctx->n_c == 2 && ctx->w_rows == 1 && ctx->precision == LL_PREC_FP64 && n_w >= 960)
        pl.WB = 128;
    pl.n_wp = (int)round_up(std::max<long long>(n_w, 1), pl.WB);
    const int n_wb = pl.n_wp / pl.WB;
    // aim at ~16 blocks per SM over the whole grid, tiles between 64 and LL_FUSED_TB_MAX bins.  Small batches (blocks of one
    // warp, most tiles beyond the walkers' bands and exiting at once): 8x as many, smaller tiles, so that the active
    // ones still fill the SMs (measured on 160 walkers x 1.57e6 bins: TB 4096 -> 512 halves the fused kernel's time)
    static const int small_factor = getenv("LL_SMALL_TILE_FACTOR") ? atoi(getenv("LL_SMALL_TILE_FACTOR")) : 128;
    const long long target = (long long)ctx->sm_count * (pl.n_wp <= 1024 ? small_factor : 16);
    long long tb = ctx->n_f * n_wb / target;
    int TB = 64;
#ifndef LL_SMALL_CH
#define LL_SMALL_CH 128 // bins per TMA stage of the one-warp blocks of small batches (10 KB per block, 16 blocks per SM); 160 walkers on the config-2 grid: 32 bins 0.183 ms, 64: 0.161, 96: 0.153, 128: 0.151, 160: 0.152, 192 and 256 (fewer resident blocks): 0.179
#endif
#ifndef LL_FUSED_TB_MAX
#define LL_FUSED_TB_MAX 2048 // config 2: 4096-bin tiles 8.92 ms (step 9.59), 2048: 8.85 (9.54), 1024: 8.81 (9.53), 512: 8.91 (9.68)
#endif
    while (TB < LL_FUSED_TB_MAX && TB < tb) TB <<= 1;
    pl.TB = TB;
    // bins per TMA stage: blocks of one warp (small batches) take 64-bin stages, 5 KB of shared memory per block, so
    // that shared memory does not hold an SM to 11 resident warps (ncu r02a: 12 % warps active with 256-bin stages)
    // (other layouts keep 256-bin stages: with 9 doubles per bin two 512-bin stages would pass the 48 KB a launch gets
    // without opting in, and hold an SM to three blocks;
    // and the multi-mode kernel measured 24.8 ms with 256-bin stages against 28.0 ms with 512 at six modes)
    constexpr int mid_ch = 256; // 64-walker blocks (exactly 1024 walkers that do not take the small route)
    pl.CH = std::min(TB, pl.WB == 32 ? LL_SMALL_CH : ((ctx->n_c == 2 && ctx->w_rows == 1 && ctx->n_m == 1) ? (pl.WB == 64 ? mid_ch : LL_FUSED_CH) : 256));
    pl.n_tiles = ceil_div(ctx->n_f, TB);
    pl.key_gran = std::max(1, ceil_div(ctx->n_f, 4096));
    pl.n_keys = (int)(ctx->n_f / pl.key_gran) + 2;
    return pl;
}

// Frequency tiles of the fused kernel.  Large batches: uniform tiles of TB bins.  Small batches (latency matters:
// Module-1 sized): a tile is also limited by the spline intervals it crosses, since every interval
// change costs one dependent global load of the coefficients (~14 bins' worth of arithmetic) and log-spaced nodes
// put dozens of intervals into the first tiles of the grid; cost = bins + 14 per interval <= TB.
constexpr int kTileChunk = 64;
// work items of the small-batch fused kernel per SM (16 one-warp blocks are resident per SM, by registers).  160 walkers on the
// config-2 grid with lanes items: 12 per SM 0.161 ms, 16: 0.129, 20: 0.138, 24: 0.1249, 28: 0.1249, 32: 0.1254, 48: 0.1265, 64: 0.128
// (the plan and F4 grow with the item count: whole call 0.1705 at 16, 0.1667 at 24, 0.175 at 48)
constexpr int kSmallWarpsPerSM = 24;
int ensure_tiles(ll_ctx *ctx, FullPlan &pl, cudaStream_t st, bool uniform = false)
{
    const int small = uniform ? 2 : (pl.n_wp <= 1024 ? 1 : 0); // 2: per-walker node grids, no shared interval table
    ll_ctx::TileCache &tc = ctx->tiles[small];
    ctx->tile_cur = &tc;
    // kinds 0 and 2 depend on the grid only; kind 1 also on the node set (its interval table)
    if (tc.data_version == ctx->data_version && tc.TB == pl.TB && (small != 1 || tc.nodes_version == ctx->nodes_version)) {
        pl.n_tiles = tc.n;
        return LL_OK;
    }
    const int n_f = (int)ctx->n_f, n = (int)ctx->bstart_host.size();
    std::vector<int> ts;
    ts.push_back(0);
    if (small != 1) {
        for (int i = pl.TB; i < n_f; i += pl.TB) ts.push_back(i);
    } else {
        const int kIntervalCost = 14;
        int end = 0, j = 0;
        while (end < n_f) {
            int cost = 0;
            const int start = end;
            while (end < n_f) {
                while (j < n - 2 && ctx->bstart_host[j + 1] <= end) ++j;
                const int seg_end = (j < n - 2) ? ctx->bstart_host[j + 1] : n_f;
                const int room = pl.TB - cost - kIntervalCost;
                if (room <= 0 && end > start) break;
                const int take = std::min(seg_end - end, std::max(room, 1));
                end += take;
                cost += take + kIntervalCost;
            }
            ts.push_back(end);
        }
        ts.pop_back();
    }
    ts.push_back(n_f);
    pl.n_tiles = (int)ts.size() - 1;
    // chunk boundaries for the two-stage finalize of small batches: tile_start2[z] = tile_start[z * kTileChunk]
    tc.off2 = (int)ts.size();
    tc.n2 = ceil_div(pl.n_tiles, kTileChunk);
    for (int z = 0; z < tc.n2; ++z) ts.push_back(ts[(size_t)z * kTileChunk]);
    ts.push_back(n_f);
    tc.data_version = -1; // not valid until the copy below has been enqueued
    CK(tc.tab.ensure(sizeof(int) * ts.size()));
    CK(cudaMemcpyAsync(tc.tab.p, ts.data(), sizeof(int) * ts.size(), cudaMemcpyHostToDevice, st));
    CK(cudaStreamSynchronize(st)); // ts goes out of scope
    tc.data_version = ctx->data_version;
    tc.nodes_version = ctx->nodes_version;
    tc.TB = pl.TB;
    tc.n = pl.n_tiles;
    return LL_OK;
}

// band -> bin range per walker, sort by band top (F1 prologue shared by every full-grid entry point)
// defer: (batches of up to 1024 walkers) fill the planner's arguments instead of launching it — the caller runs it as the
// last block of k_setup_small
int band_sort(ll_ctx *ctx, const FullPlan &pl, long long n_w, bool standin, const double *params, int P, const double *band,
              cudaStream_t st, int n_items = 0, BandSortArgs *defer = nullptr, bool allow_lanes = true, bool shared_nodes = true)
{
    const int n_wp = pl.n_wp;
    CK(ctx->ilo_w.ensure(sizeof(int) * n_wp));
    CK(ctx->ihi_w.ensure(sizeof(int) * n_wp));
    CK(ctx->key_w.ensure(sizeof(int) * 2 * n_wp)); // keys, then the unordered buckets
    CK(ctx->perm.ensure(sizeof(int) * n_wp));
    CK(ctx->ilo_s.ensure(sizeof(int) * n_wp));
    CK(ctx->ihi_s.ensure(sizeof(int) * n_wp));
    CK(ctx->hist.ensure(sizeof(int) * (2 * 8192 + 1))); // cursors, then the bucket starts
    CK(ctx->pairs.ensure(sizeof(unsigned long long)));
    const GridInfo g{ctx->k_min, ctx->n_f, ctx->df};
    if (n_w <= 1024 && n_wp <= 1024) {
        // = the fused kernel's grid: rounding gives every live group at least one group item (up to 32 more than n_items)
        // and every walker's lanes items one more than its share (up to n_wp more)
        const int max_items = n_items ? n_items + 32 + n_wp : 0;
        if (n_items) CK(ctx->grp_tab.ensure(sizeof(int) * (grp_off_items() + 4 * (size_t)max_items)));
        BandSortArgs ba;
        ba.use_standin = standin ? 1 : 0; ba.params = params; ba.P = P; ba.band = band; ba.n_w = (int)n_w; ba.n_wp = n_wp;
        ba.g = g; ba.si = ctx->si; ba.perm = ctx->perm.as<int>(); ba.ilo_s = ctx->ilo_s.as<int>(); ba.ihi_s = ctx->ihi_s.as<int>();
        ba.pairs = ctx->pairs.as<unsigned long long>(); ba.n_items = n_items; ba.max_items = max_items;
        ba.grp_tab = n_items ? ctx->grp_tab.as<int>() : nullptr;
        ba.bstart_g = (n_items && shared_nodes) ? ctx->nt.bstart : nullptr; // per-walker node grids: no shared interval table
        ba.n_nodes = shared_nodes ? (int)ctx->nodes_host.size() : 0;
        ba.lanes = (allow_lanes && shared_nodes && ctx->n_m == 1 && ctx->precision == LL_PREC_FP64) ? 1 : 0; // the single-mode kernels
        if (defer) {
            *defer = ba;
            return LL_OK;
        }
        k_band_sort_small<<<1, 1024, 0, st>>>(ba);
        LAUNCHED(ctx);
    } else {
        CK(cudaMemsetAsync(ctx->hist.p, 0, sizeof(int) * pl.n_keys, st));
        CK(cudaMemsetAsync(ctx->pairs.p, 0, sizeof(unsigned long long), st));
        k_band_prep<<<ceil_div(n_w, 256), 256, 0, st>>>(standin ? 1 : 0, params, P, band, (int)n_w, g, ctx->si, pl.key_gran,
                                                        ctx->ilo_w.as<int>(), ctx->ihi_w.as<int>(), ctx->key_w.as<int>(),
                                                        ctx->hist.as<int>(), ctx->pairs.as<unsigned long long>());
        LAUNCHED(ctx);
        int *starts = ctx->hist.as<int>() + 8192, *bucket = ctx->key_w.as<int>() + n_wp;
        k_scan_hist<<<1, 1024, 0, st>>>(ctx->hist.as<int>(), pl.n_keys, starts);
        LAUNCHED(ctx);
        k_scatter<<<ceil_div(n_w, 256), 256, 0, st>>>((int)n_w, ctx->key_w.as<int>(), ctx->hist.as<int>(), bucket);
        LAUNCHED(ctx);
        k_sort_buckets<<<pl.n_keys + 1, kSortThreads, 0, st>>>((int)n_w, n_wp, pl.n_keys, starts, bucket, ctx->key_w.as<int>(),
                                                               ctx->ilo_w.as<int>(), ctx->ihi_w.as<int>(), ctx->perm.as<int>(),
                                                               ctx->ilo_s.as<int>(), ctx->ihi_s.as<int>());
        LAUNCHED(ctx);
    }
    return LL_OK;
}

FusedArgs fused_args(ll_ctx *ctx, const FullPlan &pl, int n_nodes, const double *t_shift, int ts_stride)
{
    FusedArgs fa;
    fa.g = ctx->g.as<double>(); fa.Wc = ctx->Wc.as<double>(); fa.C = ctx->C.as<double>(); fa.TF = ctx->TF.as<double>();
    fa.xj = ctx->nt.xj; fa.bstart = ctx->nt.bstart; fa.ilo = ctx->ilo_s.as<int>(); fa.ihi = ctx->ihi_s.as<int>();
    fa.perm = ctx->perm.as<int>(); fa.t_shift = t_shift; fa.ts_stride = ts_stride;
    fa.part = ctx->part.as<double>(); fa.k_min = ctx->k_min; fa.n_f_pad = ctx->n_f_pad; fa.df = ctx->df;
    fa.n_f = (int)ctx->n_f; fa.n_wp = pl.n_wp; fa.n_nodes = n_nodes; fa.n_m = ctx->n_m; fa.TB = pl.TB; fa.CH = pl.CH;
    fa.tile_start = ctx->tile_cur ? ctx->tile_cur->tab.as<int>() : nullptr;
    fa.grp_tab = ctx->grp_tab.as<int>();
    fa.wmom = (ctx->precision == LL_PREC_FP64 && ctx->n_m == 1) ? ctx->wmom.as<double>() : nullptr;
    return fa;
}

// F4: partial sums over tiles (two stages for small batches with thousands of tiles) -> log L
int finalize(ll_ctx *ctx, const FullPlan &pl, bool single_mode_sums, double *logL, double *d_h, double *h_h, cudaStream_t st)
{
    const int n_wp = pl.n_wp, n_c = ctx->n_c, nw = ctx->w_rows;
    const int NQ = single_mode_sums ? 2 * n_c + nw : 2;
    const double *fin_part = ctx->part.as<double>();
    const int *fin_tiles = ctx->tile_cur->tab.as<int>();
    int fin_n = pl.n_tiles;
    if (n_wp <= 1024 && pl.n_tiles >= 8 * kTileChunk) { // thousands of tiles, a handful of walker blocks: two stages
        CK(ctx->part2.ensure(sizeof(double) * (size_t)ctx->tile_cur->n2 * NQ * n_wp));
        dim3 grid(ceil_div(n_wp, 32), ctx->tile_cur->n2);
#define LL_REDUCE(Q)                                                                                                     \
    k_reduce_tiles<Q><<<grid, dim3(32, fin_slices(Q)), 0, st>>>(fin_part, ctx->ilo_s.as<int>(), ctx->ihi_s.as<int>(), n_wp, fin_tiles, \
                                                     fin_n, kTileChunk, ctx->part2.as<double>())
        switch (NQ) {
        case 2: LL_REDUCE(2); break;
        case 5: LL_REDUCE(5); break;
        case 6: LL_REDUCE(6); break;
        default: LL_REDUCE(9); break;
        }
#undef LL_REDUCE
        LAUNCHED(ctx);
        fin_part = ctx->part2.as<double>();
        fin_tiles = ctx->tile_cur->tab.as<int>() + ctx->tile_cur->off2;
        fin_n = ctx->tile_cur->n2;
    }
#define LL_FIN(NC, WS)                                                                                                    \
    do {                                                                                                                  \
        if (single_mode_sums)                                                                                             \
            k_finalize<1, NC, (WS ? 1 : NC)><<<ceil_div(n_wp, 32), dim3(32, fin_slices(2 * NC + (WS ? 1 : NC))), 0, st>>>(                             \
                fin_part, ctx->TF.as<double>(), ctx->perm.as<int>(), ctx->ilo_s.as<int>(), ctx->ihi_s.as<int>(), n_wp,    \
                fin_tiles, fin_n, ctx->dd.as<double>(), logL, d_h, h_h);                                                  \
        else                                                                                                              \
            k_finalize<0, NC, (WS ? 1 : NC)><<<ceil_div(n_wp, 32), dim3(32, fin_slices(2)), 0, st>>>(                             \
                fin_part, ctx->TF.as<double>(), ctx->perm.as<int>(), ctx->ilo_s.as<int>(), ctx->ihi_s.as<int>(), n_wp,    \
                fin_tiles, fin_n, ctx->dd.as<double>(), logL, d_h, h_h);                                                  \
    } while (0)
    LL_LAYOUT(ctx, LL_FIN);
#undef LL_FIN
    LAUNCHED(ctx);
    return LL_OK;
}

// the whole full-grid pipeline for walkers [0, n_w) given either stand-in params or caller arrays
int run_full(ll_ctx *ctx, long long n_w, int n_nodes, const double *params, const double *amp, const double *phase,
             const double *tf, const double *band, const double *t_shift, double *logL, double *d_h, double *h_h,
             cudaStream_t st, bool template_only, double *h_out, const double *tf_nodes = nullptr)
{
    const bool standin = params != nullptr;
    const bool tfp = tf_nodes != nullptr; // frequency-dependent transfer function: 2 + 2 n_c splines per mode
    const int n_m = ctx->n_m, n_c = ctx->n_c, nw = ctx->w_rows;
    const int ns = tfp ? 2 + 2 * n_c : 2;
    const int P = 5 + 2 * n_c * n_m;
    FullPlan pl = make_plan(ctx, n_w, !tfp && !template_only);
    // small batches (Module-1 sized): blocks of one warp, the work dealt out by active bins (k_band_sort_small)
    // (the T(f) entry point too: 160 walkers on the one-year grid, kernel 0.397 ms on the large route's uniform tiles, 0.325 with
    // group items, 0.236 with lanes items; 1024 walkers 1.58 / 1.66 / 1.47)
    const bool small = pl.n_wp <= 1024 && pl.WB != 128 && !template_only && ctx->precision == LL_PREC_FP64;
    static const int small_wps = getenv("LL_SMALL_WPS") ? atoi(getenv("LL_SMALL_WPS")) : kSmallWarpsPerSM;
    const int n_items = small ? ctx->sm_count * small_wps : 0;
    if (!small) {
        const int rc_t = ensure_tiles(ctx, pl, st);
        if (rc_t != LL_OK) return rc_t;
    }
    const int n_wp = pl.n_wp;
    const bool nm1 = (n_m == 1);
    const bool sums1 = nm1 && !tfp; // the single-mode kernel leaves S^c, H^c and k_finalize applies T^c
    const int NQ = sums1 ? 2 * n_c + nw : 2;
    int ts_stride = 1;
    if (standin && ctx->si.split_tc) { t_shift = params + 2; ts_stride = P; } // the stand-in's own linear term (R32)

    CK(ctx->Y.ensure(sizeof(double) * (size_t)n_m * ns * n_nodes * n_wp));
    CK(ctx->C.ensure(sizeof(double) * (size_t)(n_nodes - 1) * n_m * ns * 4 * n_wp));
    CK(ctx->TF.ensure(sizeof(double) * (size_t)n_m * 2 * n_c * n_wp));
    if (small) CK(ctx->part.ensure(sizeof(double) * (size_t)(n_items + 32 + pl.n_wp) * NQ * 32));
    else if (!template_only) CK(ctx->part.ensure(sizeof(double) * (size_t)pl.n_tiles * NQ * n_wp));
    // few systems (Module-1 sized batches): a block per four walkers of a system, scan-based sweeps (k_spline_block4), and on
    // the stand-in path the block evaluates its own node values (no k_nodes_standin launch, no Y); else one thread per system
    const long long n_sys = (long long)n_wp * ns * n_m;
    // measured on 160 walkers x 1024 nodes (whole call): 1 walker per block 0.2095 ms (256 threads), 2: 0.2056 (512),
    // 4: 0.2014 (512 or 1024 threads; 0.2054 with 256) — latency-bound: ~2000 dependent instructions per warp whatever the shape
    constexpr int NWK4 = 4; // walkers per block of k_spline_block4
    int T4 = 32 * NWK4;     // its threads: NWK4 walkers x ~8 rows per chunk thread, at most 512
    while (T4 < 512 && T4 < n_nodes * NWK4 / 8) T4 <<= 1;
    const size_t smem4 = sizeof(double) * (2 * (size_t)NWK4 * n_nodes + T4);
    const bool block4 = n_sys <= (long long)ctx->sm_count * 32 && smem4 <= 160 * 1024;
    if (block4 && !ctx->spl4_attr) {
#define LL_SPL4_ATTR(S, N) CK(cudaFuncSetAttribute(k_spline_block4<S, N>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024))
        LL_SPL4_ATTR(true, NWK4);
        LL_SPL4_ATTR(false, NWK4);
#undef LL_SPL4_ATTR
        CK(cudaFuncSetAttribute(k_setup_small<NWK4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024));
        ctx->spl4_attr = true;
    }
    // stand-in batches of up to 1024 walkers: planner, F1 and F2 in one launch (k_setup_small)
    // (up to 512 walkers: every spline block ranks all walkers itself, O(n_w) per thread — measured whole call, merged against
    // separate launches: 160 walkers 0.167 / 0.190 ms, 320: 0.287 / 0.298, 480: 0.444 / 0.453, 640: 0.605 / 0.587, 1024: 1.00 / 0.91)
    const bool merged = standin && block4 && n_w <= 512 && n_wp <= 1024 &&
                        sizeof(double) * (2 * (size_t)NWK4 * n_nodes + 1024) <= 160 * 1024;
    BandSortArgs ba;
    {
        const int rc_b = band_sort(ctx, pl, n_w, standin, params, P, band, st, n_items, merged ? &ba : nullptr);
        if (rc_b != LL_OK) return rc_b;
    }
    Spline4Args sa;
    sa.Y = standin ? nullptr : ctx->Y.as<double>(); sa.C = ctx->C.as<double>(); sa.n_wp = n_wp; sa.n_nodes = n_nodes; sa.n_m = n_m;
    sa.ns = ns; sa.nt = ctx->nt; sa.params = params; sa.P = P; sa.perm = ctx->perm.as<int>(); sa.si = ctx->si;
    sa.TF = ctx->TF.as<double>();
    if (standin && block4) {
        // F1 happens inside F2 (below)
    } else if (standin) {
        dim3 grid(ceil_div(n_wp, 128), ceil_div(n_nodes, kNodesPerThread));
        k_nodes_standin<<<grid, 128, 0, st>>>(params, P, ctx->perm.as<int>(), n_wp, n_nodes, ctx->si, ctx->nt,
                                              ctx->Y.as<double>(), ctx->TF.as<double>());
    } else if (tfp) {
        dim3 grid(n_wp / 32, ceil_div(n_nodes, 32), n_m * ns);
        k_nodes_arrays_tf<<<grid, 256, 0, st>>>(amp, phase, tf_nodes, ctx->perm.as<int>(), n_wp, n_nodes, n_m, n_c,
                                                ctx->Y.as<double>());
    } else {
        dim3 grid(n_wp / 32, ceil_div(n_nodes, 32), n_m);
        k_nodes_arrays<<<grid, 256, 0, st>>>(amp, phase, tf, ctx->perm.as<int>(), n_wp, n_nodes, n_m, n_c,
                                             ctx->Y.as<double>(), ctx->TF.as<double>());
    }
    if (!(standin && block4)) LAUNCHED(ctx);
    {
        if (merged) {
            const size_t smem_m = sizeof(double) * (2 * (size_t)NWK4 * n_nodes + 1024);
            k_setup_small<NWK4><<<(unsigned)(n_sys / NWK4) + 1, 1024, smem_m, st>>>(sa, ba);
        } else if (block4) {
            if (standin) k_spline_block4<true, NWK4><<<(unsigned)(n_sys / NWK4), T4, smem4, st>>>(sa);
            else k_spline_block4<false, NWK4><<<(unsigned)(n_sys / NWK4), T4, smem4, st>>>(sa);
        } else {
            dim3 grid(ceil_div(n_wp, 128), ns * n_m);
            k_spline<<<grid, 128, 0, st>>>(ctx->Y.as<double>(), ctx->C.as<double>(), n_wp, n_nodes, n_m, ns, ctx->nt);
        }
        LAUNCHED(ctx);
    }
    const FusedArgs fa = fused_args(ctx, pl, n_nodes, t_shift, ts_stride);
    if (template_only) {
        // sorted position of walker 0 of a one-walker batch is 0
        k_full_template<<<ceil_div(ctx->n_f, 256), 256, 0, st>>>(fa, 0, n_c, h_out);
        LAUNCHED(ctx);
        return LL_OK;
    }
    if (small) {
        const int grid = n_items + 32 + n_wp; // = max_items of the planner (band_sort)
        // three or six modes, the BASELINE layout: every mode by its own recurrence (k_full_fused_hm in item form)
        const int hm_small = (!nm1 && !tfp && n_c == 2 && nw == 1 && (n_m == 3 || n_m == 6)) ? n_m : 0;
        const size_t smem_hms = (size_t)2 * pl.CH * 8 * (2 * n_c + nw) + sizeof(double) * (size_t)n_m * (3 + 2 * n_c) * 32;
        const size_t smem = (size_t)2 * pl.CH * 8 * (2 * n_c + nw);
        {
            ProfScope prof(ctx, st);
#define LL_FUSED_SMALL(NC, WS)                                                        \
    do {                                                                              \
        if (tfp) {                                                                    \
            if (nm1) k_full_fused_tf<1, NC, WS, 1><<<grid, 32, smem, st>>>(fa);       \
            else k_full_fused_tf<0, NC, WS, 1><<<grid, 32, smem, st>>>(fa);           \
        } else if (nm1) k_full_fused<1, NC, WS, 1><<<grid, 32, smem, st>>>(fa);       \
        else if (hm_small == 6) k_full_fused_hm<6, 2, true, 1><<<grid, 32, smem_hms, st>>>(fa); \
        else if (hm_small == 3) k_full_fused_hm<3, 2, true, 1><<<grid, 32, smem_hms, st>>>(fa); \
        else k_full_fused<0, NC, WS, 1><<<grid, 32, smem, st>>>(fa);                  \
    } while (0)
            LL_LAYOUT(ctx, LL_FUSED_SMALL);
#undef LL_FUSED_SMALL
            LAUNCHED(ctx);
        }
        ctx->last_n_blocks = grid;
        CK(ctx->part2.ensure(sizeof(double) * (size_t)(n_wp / 32) * kFinZ * 9 * 32)); // [group][kFinZ][NQ <= 9][32]
#define LL_FIN_SMALL(NC, WS)                                                                                               \
    do {                                                                                                                   \
        if (sums1)                                                                                                         \
            k_finalize_small<1, NC, (WS ? 1 : NC)><<<dim3(n_wp / 32, kFinZ), dim3(32, fin_slices(2 * NC + (WS ? 1 : NC))), 0, st>>>( \
                ctx->part.as<double>(), ctx->part2.as<double>(), ctx->TF.as<double>(), ctx->perm.as<int>(), n_wp,          \
                ctx->grp_tab.as<int>(), ctx->dd.as<double>(), logL, d_h, h_h);                                             \
        else                                                                                                               \
            k_finalize_small<0, NC, (WS ? 1 : NC)><<<dim3(n_wp / 32, kFinZ), dim3(32, fin_slices(2)), 0, st>>>(            \
                ctx->part.as<double>(), ctx->part2.as<double>(), ctx->TF.as<double>(), ctx->perm.as<int>(), n_wp,          \
                ctx->grp_tab.as<int>(), ctx->dd.as<double>(), logL, d_h, h_h);                                             \
    } while (0)
        LL_LAYOUT(ctx, LL_FIN_SMALL);
#undef LL_FIN_SMALL
        LAUNCHED(ctx);
        return LL_OK;
    }
    {
        dim3 grid(n_wp / pl.WB, pl.n_tiles);
        const bool mixed = ctx->precision == LL_PREC_FP32_ACC && !tfp;
        const size_t smem = (size_t)2 * pl.CH * (mixed ? 24 : 8 * (2 * n_c + nw));
        // several modes, the BASELINE layout, FP64, blocks of 128 walkers: the recurrence kernel (instantiated for 3 and 6 modes)
        const int hm_rot = (!nm1 && !tfp && !mixed && ctx->precision == LL_PREC_FP64 && n_c == 2 && nw == 1 && pl.WB == 128 &&
                            (n_m == 3 || n_m == 6)) ? n_m : 0;
        const size_t smem_hm = smem + sizeof(double) * (size_t)n_m * (3 + 2 * n_c) * 128;
        if (hm_rot && !ctx->hm_attr) {
            CK(cudaFuncSetAttribute(k_full_fused_hm<6, 2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
            CK(cudaFuncSetAttribute(k_full_fused_hm<3, 2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
            ctx->hm_attr = true;
        }
        ProfScope prof(ctx, st);
        if (mixed) {
            const FusedArgsF32 fm{ctx->g4f.as<float>(), ctx->Wf.as<double>(), ctx->scale.as<double>()};
            k_full_fused_mixed<<<grid, pl.WB, smem, st>>>(fa, fm);
        } else {
#define LL_FUSED(NC, WS)                                                              \
    do {                                                                              \
        if (tfp) {                                                                    \
            if (nm1) k_full_fused_tf<1, NC, WS><<<grid, pl.WB, smem, st>>>(fa);       \
            else k_full_fused_tf<0, NC, WS><<<grid, pl.WB, smem, st>>>(fa);           \
        } else if (nm1) k_full_fused<1, NC, WS, 0><<<grid, pl.WB, smem, st>>>(fa);    \
        else if (hm_rot == 6) k_full_fused_hm<6, 2, true><<<grid, pl.WB, smem_hm, st>>>(fa); \
        else if (hm_rot == 3) k_full_fused_hm<3, 2, true><<<grid, pl.WB, smem_hm, st>>>(fa); \
        else k_full_fused<0, NC, WS, 0><<<grid, pl.WB, smem, st>>>(fa);               \
    } while (0)
            LL_LAYOUT(ctx, LL_FUSED);
#undef LL_FUSED
        }
        LAUNCHED(ctx);
        ctx->last_n_blocks = (int)(grid.x * grid.y);
    }
    return finalize(ctx, pl, sums1, logL, d_h, h_h, st);
}

// full-grid pipeline with per-walker node grids (reading R30)
int run_full_pw(ll_ctx *ctx, long long n_w, int n_nodes, const double *f_nodes_w, const double *amp, const double *phase,
                const double *tf, const double *band, const double *t_shift, double *logL, double *d_h, double *h_h,
                cudaStream_t st)
{
    const int n_m = ctx->n_m, n_c = ctx->n_c, nw = ctx->w_rows;
    FullPlan pl = make_plan(ctx, n_w);
    // small batches: one-warp blocks over the planner's group items (as run_full), the split F4
    const bool small = pl.n_wp <= 1024 && pl.WB != 128 && ctx->precision == LL_PREC_FP64;
    const int n_items = small ? ctx->sm_count * kSmallWarpsPerSM : 0;
    if (!small) {
        const int rc_t = ensure_tiles(ctx, pl, st, true);
        if (rc_t != LL_OK) return rc_t;
    }
    const int n_wp = pl.n_wp;
    const int NQ = 2;
    CK(ctx->Y.ensure(sizeof(double) * (size_t)n_m * 2 * n_nodes * n_wp));
    CK(ctx->C.ensure(sizeof(double) * (size_t)(n_nodes - 1) * n_m * 8 * n_wp));
    CK(ctx->TF.ensure(sizeof(double) * (size_t)n_m * 2 * n_c * n_wp));
    if (small) CK(ctx->part.ensure(sizeof(double) * (size_t)(n_items + 32 + n_wp) * NQ * 32));
    else CK(ctx->part.ensure(sizeof(double) * (size_t)pl.n_tiles * NQ * n_wp));
    CK(ctx->pw_x.ensure(sizeof(double) * ((size_t)n_nodes * n_wp + 2 * (size_t)n_w)));
    double *X = ctx->pw_x.as<double>(), *band_w = X + (size_t)n_nodes * n_wp;

    k_pw_band<<<ceil_div(n_w, 256), 256, 0, st>>>(f_nodes_w, band, (int)n_w, n_nodes, band_w);
    LAUNCHED(ctx);
    {
        const int rc_b = band_sort(ctx, pl, n_w, false, nullptr, 0, band_w, st, n_items, nullptr, false, false);
        if (rc_b != LL_OK) return rc_b;
    }
    {
        dim3 grid(n_wp / 32, ceil_div(n_nodes, 32), n_m);
        k_nodes_arrays<<<grid, 256, 0, st>>>(amp, phase, tf, ctx->perm.as<int>(), n_wp, n_nodes, n_m, n_c, ctx->Y.as<double>(),
                                             ctx->TF.as<double>());
        LAUNCHED(ctx);
        dim3 gx(n_wp / 32, ceil_div(n_nodes, 32));
        k_pw_nodes_x<<<gx, 256, 0, st>>>(f_nodes_w, ctx->perm.as<int>(), n_wp, n_nodes, X);
        LAUNCHED(ctx);
        // few systems (Module-1 sized batches): a block per four walkers of a system (k_spline_pw_block); else a thread per system
        const long long n_sys = (long long)n_wp * 2 * n_m;
        int Tb = 128;
        while (Tb < 512 && Tb < n_nodes / 2) Tb <<= 1; // four walkers x ~8 rows per chunk thread
        const size_t smem_b = sizeof(double) * (16 * (size_t)n_nodes + Tb);
        if (n_sys <= (long long)ctx->sm_count * 32 && smem_b <= 160 * 1024 && n_nodes >= 4) {
            if (!ctx->splpw_attr) {
                CK(cudaFuncSetAttribute(k_spline_pw_block<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024));
                ctx->splpw_attr = true;
            }
            k_spline_pw_block<4><<<(unsigned)(n_sys / 4), Tb, smem_b, st>>>(ctx->Y.as<double>(), X, ctx->C.as<double>(), n_wp, n_nodes,
                                                                            n_m, ctx->spline_bc);
        } else {
            dim3 gs(ceil_div(n_wp, 128), 2 * n_m);
            k_spline_pw<<<gs, 128, 0, st>>>(ctx->Y.as<double>(), X, ctx->C.as<double>(), n_wp, n_nodes, n_m, ctx->spline_bc);
        }
        LAUNCHED(ctx);
    }
    FusedArgs fa = fused_args(ctx, pl, n_nodes, t_shift, 1);
    fa.xj = nullptr; fa.bstart = nullptr;
    if (small) {
        const int grid = n_items + 32 + n_wp; // = max_items of the planner
        const size_t smem = (size_t)2 * pl.CH * 8 * (2 * n_c + nw);
        {
            ProfScope prof(ctx, st);
#define LL_FUSED_PW_SMALL(NC, WS)                                                          \
    do {                                                                                   \
        if (n_m == 1) k_full_fused_pw<1, NC, WS, 1><<<grid, 32, smem, st>>>(fa, X);        \
        else k_full_fused_pw<0, NC, WS, 1><<<grid, 32, smem, st>>>(fa, X);                 \
    } while (0)
            LL_LAYOUT(ctx, LL_FUSED_PW_SMALL);
#undef LL_FUSED_PW_SMALL
            LAUNCHED(ctx);
        }
        ctx->last_n_blocks = grid;
        CK(ctx->part2.ensure(sizeof(double) * (size_t)(n_wp / 32) * kFinZ * 9 * 32));
#define LL_FIN_PW_SMALL(NC, WS)                                                                                            \
    k_finalize_small<0, NC, (WS ? 1 : NC)><<<dim3(n_wp / 32, kFinZ), dim3(32, fin_slices(2)), 0, st>>>(                    \
        ctx->part.as<double>(), ctx->part2.as<double>(), ctx->TF.as<double>(), ctx->perm.as<int>(), n_wp, ctx->grp_tab.as<int>(), \
        ctx->dd.as<double>(), logL, d_h, h_h)
        LL_LAYOUT(ctx, LL_FIN_PW_SMALL);
#undef LL_FIN_PW_SMALL
        LAUNCHED(ctx);
        return LL_OK;
    }
    {
        dim3 grid(n_wp / pl.WB, pl.n_tiles);
        const size_t smem = (size_t)2 * pl.CH * 8 * (2 * n_c + nw);
        ProfScope prof(ctx, st);
#define LL_FUSED_PW(NC, WS)                                                            \
    do {                                                                               \
        if (n_m == 1) k_full_fused_pw<1, NC, WS><<<grid, pl.WB, smem, st>>>(fa, X);    \
        else k_full_fused_pw<0, NC, WS><<<grid, pl.WB, smem, st>>>(fa, X);             \
    } while (0)
        LL_LAYOUT(ctx, LL_FUSED_PW);
#undef LL_FUSED_PW
        LAUNCHED(ctx);
        ctx->last_n_blocks = (int)(grid.x * grid.y);
    }
    return finalize(ctx, pl, false, logL, d_h, h_h, st);
}

int check_full_common(ll_ctx *ctx, int64_t n_w, const double *f_nodes, const double *logL)
{
    if (!ctx) return LL_ERR_ARG;
    if (n_w < 0) return ctx->fail(LL_ERR_ARG, "n_w < 0");
    if (n_w > (1 << 24)) return ctx->fail(LL_ERR_ARG, "n_w > 2^24 per call: split the batch");
    if (!f_nodes) return ctx->fail(LL_ERR_ARG, "f_nodes is NULL");
    if (n_w > 0 && !logL) return ctx->fail(LL_ERR_ARG, "logL is NULL");
    if (!ctx->have_data) return ctx->fail(LL_ERR_STATE, "ll_set_data has not been called");
    if (ctx->precision == LL_PREC_FP32_ACC && (ctx->n_m != 1 || ctx->n_c != 2 || ctx->w_rows != 1))
        return ctx->fail(LL_ERR_UNSUPPORTED, "the FP32-accumulate variant is built for n_modes = 1, two channels, one shared weight row only");
    return LL_OK;
}

// packed heterodyne table on the host
int build_het_table(ll_ctx *ctx, int n_e, const double *e, const std::vector<double> &h0e, std::vector<double> &tab)
{
    typedef long double ld;
    const int n_b = n_e - 1, n_m = ctx->n_m, n_c = ctx->n_c, NR = 6 * n_c + 1;
    HetTable T;
    T.base = nullptr; T.n_e = n_e; T.n_b = n_b; T.n_m = n_m; T.n_c = n_c;
    T.total = (1 + 2 * n_c) * n_e + 3 * n_m * n_e + 6 * n_c * n_b;
    tab.assign(T.total, 0.0);
    for (int j = 0; j < n_e; ++j) {
        tab[T.off_f4() + j] = 4.0 * e[j];
        for (int c = 0; c < n_c; ++c) {
            const ld gr = h0e[((size_t)c * n_e + j) * 2], gi = h0e[((size_t)c * n_e + j) * 2 + 1];
            const ld den = gr * gr + gi * gi;
            if (!(den > 0.0L) || !std::isfinite((double)den)) return ctx->fail(LL_ERR_REF_ZERO, "h0 is zero or non-finite at a bin edge");
            tab[T.off_ih0() + 2 * n_c * j + 2 * c] = (double)(gr / den);
            tab[T.off_ih0() + 2 * n_c * j + 2 * c + 1] = (double)(-gi / den);
        }
        if (ctx->have_standin)
            for (int m = 0; m < n_m; ++m) {
                const ld f = (ld)e[j], fp = 2.0L * f / (ld)ctx->si.mode_m[m];
                tab[T.off_cfp() + m * n_e + j] = (double)((ld)ctx->c_lm[m] * powl(f, -7.0L / 6.0L));
                tab[T.off_f2m() + m * n_e + j] = (double)fp;
                // (m / pi) (2f/m)^(-5/3): the mode's phase factor m/2 and the radians -> quarter cycles 2/pi folded in
                tab[T.off_fm53() + m * n_e + j] = (double)((ld)ctx->si.mode_m[m] / 3.14159265358979323846264338327950288L *
                                                           powl(fp, -5.0L / 3.0L));
            }
    }
    const std::vector<double> &raw = ctx->raw_host;
    for (int b = 0; b < n_b; ++b) {
        const ld invw = 1.0L / ((ld)e[b + 1] - (ld)e[b]);
        double *t = &tab[T.off_bins() + 6 * n_c * b];
        // raw: per channel (A0r, A0i, A1r, A1i, B0, B1); table: A0/2 [2 n_c], A1/width [2 n_c], B0/4 [n_c], B1/width [n_c]
        for (int c = 0; c < n_c; ++c) {
            const double *r = &raw[(size_t)b * NR + 6 * c];
            t[2 * c] = 0.5 * r[0]; t[2 * c + 1] = 0.5 * r[1];
            t[2 * n_c + 2 * c] = (double)((ld)r[2] * invw); t[2 * n_c + 2 * c + 1] = (double)((ld)r[3] * invw);
            t[4 * n_c + c] = 0.25 * r[4];
            t[5 * n_c + c] = (double)((ld)r[5] * invw);
        }
    }
    ctx->ht = T;
    return LL_OK;
}

// single-mode regrouped table (k_het_standin1): 4 + 5 n_c doubles per edge, see ll_kernels.cuh
void build_het1_table(ll_ctx *ctx, int n_e, const double *e, const std::vector<double> &h0e, std::vector<double> &tab)
{
    typedef long double ld;
    const int n_b = n_e - 1, n_c = ctx->n_c, NR = 6 * n_c + 1, ST = het1_stride(n_c);
    const int oQ = 4, oP = 4 + 2 * n_c, oX = 4 + 3 * n_c;
    const std::vector<double> &raw = ctx->raw_host; // [n_b][6 n_c + 1]: per channel (A0r, A0i, A1r, A1i, B0, B1), then dd
    tab.assign((size_t)n_e * ST, 0.0);
    std::vector<ld> ihr((size_t)n_c * n_e), ihi((size_t)n_c * n_e);
    for (int c = 0; c < n_c; ++c)
        for (int j = 0; j < n_e; ++j) {
            const ld gr = h0e[((size_t)c * n_e + j) * 2], gi = h0e[((size_t)c * n_e + j) * 2 + 1];
            const ld den = gr * gr + gi * gi;
            ihr[(size_t)c * n_e + j] = gr / den;
            ihi[(size_t)c * n_e + j] = -gi / den;
        }
    for (int j = 0; j < n_e; ++j) {
        double *t = &tab[(size_t)j * ST];
        const ld f = (ld)e[j], fp = 2.0L * f / (ld)ctx->si.mode_m[0];
        t[0] = 4.0 * e[j];
        t[1] = (double)powl(fp, -5.0L / 3.0L);
        t[2] = (double)((ld)ctx->c_lm[0] * powl(f, -7.0L / 6.0L));
        t[3] = (double)fp;
        for (int c = 0; c < n_c; ++c) {
            ld Gr = 0, Gi = 0, Pc = 0;
            if (j >= 1) { // bin j - 1 ends at this edge
                const double *r = &raw[(size_t)(j - 1) * NR + 6 * c];
                const ld invw = 1.0L / ((ld)e[j] - (ld)e[j - 1]);
                Gr += 0.5L * r[0] + r[2] * invw; Gi += 0.5L * r[1] + r[3] * invw;
                Pc += 0.25L * r[4] + r[5] * invw;
            }
            if (j < n_b) { // bin j starts at this edge
                const double *r = &raw[(size_t)j * NR + 6 * c];
                const ld invw = 1.0L / ((ld)e[j + 1] - (ld)e[j]);
                Gr += 0.5L * r[0] - r[2] * invw; Gi += 0.5L * r[1] - r[3] * invw;
                Pc += 0.25L * r[4] - r[5] * invw;
            }
            const ld ar = ihr[(size_t)c * n_e + j], ai = ihi[(size_t)c * n_e + j];
            // Q = G conj(1/h0)
            t[oQ + 2 * c] = (double)(Gr * ar + Gi * ai);
            t[oQ + 2 * c + 1] = (double)(Gi * ar - Gr * ai);
            t[oP + c] = (double)(Pc * (ar * ar + ai * ai));
            if (j < n_b) { // X = (B0/2) (1/h0_j) conj(1/h0_{j+1})
                const ld br = ihr[(size_t)c * n_e + j + 1], bi = ihi[(size_t)c * n_e + j + 1];
                const ld hb = 0.5L * raw[(size_t)j * NR + 6 * c + 4];
                t[oX + 2 * c] = (double)(hb * (ar * br + ai * bi));
                t[oX + 2 * c + 1] = (double)(hb * (ai * br - ar * bi));
            }
        }
    }
}

int het_check(ll_ctx *ctx, int64_t n_w, const double *logL)
{
    if (!ctx) return LL_ERR_ARG;
    if (n_w < 0) return ctx->fail(LL_ERR_ARG, "n_w < 0");
    if (n_w > (1LL << 30)) return ctx->fail(LL_ERR_ARG, "n_w too large");
    if (n_w > 0 && !logL) return ctx->fail(LL_ERR_ARG, "logL is NULL");
    if (!ctx->have_data) return ctx->fail(LL_ERR_STATE, "ll_set_data has not been called");
    if (!ctx->have_het) return ctx->fail(LL_ERR_STATE, "ll_het_prepare has not been called");
    return LL_OK;
}

// single mode: the regrouped kernel (one table copy per block, WY warps = G walker groups x S edge segments)
template <int NC>
int launch_het_standin1(ll_ctx *ctx, int64_t n_w, const double *params, double *logL, double *d_h, double *h_h,
                        cudaStream_t st)
{
    const int n_groups = ceil_div(n_w, 32), n_e = ctx->ht1.n_e;
    constexpr int WY = LL_HET1_WY;
    const size_t tab_d = (size_t)n_e * het1_stride(NC);
    const size_t smem = sizeof(double) * (tab_d + (tab_d & 1) + (size_t)WY * 32 * 3 * NC);
    if (!ctx->het1_attr) {
        CK(cudaFuncSetAttribute(k_het_standin1<NC>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        ctx->het1_attr = true;
    }
    if (smem > 227 * 1024) return ctx->fail(LL_ERR_UNSUPPORTED, "heterodyne tables exceed shared memory (too many bins)");
    if (ctx->het1_bps == 0 || ctx->het1_bps_smem != smem) {
        int bps = 0;
        CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, k_het_standin1<NC>, 32 * WY, smem));
        ctx->het1_bps = std::max(1, bps);
        ctx->het1_bps_smem = smem;
    }
    const int max_blocks = ctx->sm_count * ctx->het1_bps;
    int S = 1, grid = 1;
    double best = 1e300;
    for (int s = 1; s <= WY; ++s) {
        if (WY % s) continue;
        if (s > 1 && n_e / s < 8) break;
        const int G = WY / s;
        const long long passes = ceil_div(n_groups, G);
        const int gr = (int)std::min<long long>(passes, max_blocks);
        const double work = (double)ceil_div(gr, ctx->sm_count) * (double)ceil_div(passes, gr) * WY * (ceil_div(n_e, s) + 1.0);
        if (work < best * 0.999) { best = work; S = s; grid = gr; }
    }
    const int P = 5 + 2 * NC;
    ProfScope prof(ctx, st);
    k_het_standin1<NC><<<grid, dim3(32, WY), smem, st>>>(ctx->ht1, ctx->si, params, P, (int)n_w, n_groups, S,
                                                         ctx->dd.as<double>(), logL, d_h, h_h);
    LAUNCHED(ctx);
    return LL_OK;
}

template <int NM, int NC>
int launch_het_standin(ll_ctx *ctx, int64_t n_w, const double *params, double *logL, double *d_h, double *h_h,
                       cudaStream_t st)
{
    const int n_groups = ceil_div(n_w, 32), n_b = ctx->ht.n_b;
    constexpr int WY = LL_HET_WY; // warps per block, all sharing one table copy
    // table + [WY][2][32] segment partials + -(m/pi) + the staged parameter rows of the G = WY/S walker groups
    auto smem_of = [&](int s) { return sizeof(double) * ((size_t)ctx->ht.total + (size_t)WY * 64 + 8 + (size_t)(WY / s) * 32 * (5 + 2 * NC * NM)); };
    if (!ctx->hetn_attr) { // a context has one n_modes and one n_channels, so one instantiation
        CK(cudaFuncSetAttribute(k_het_standin<NM, NC>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        ctx->hetn_attr = true;
    }
    if (smem_of(WY) > 227 * 1024) return ctx->fail(LL_ERR_UNSUPPORTED, "heterodyne tables exceed shared memory (too many bins x modes)");
    // S = frequency segments per walker group (G = WY/S groups per block pass): pick the split whose busiest SM
    // has the least work, work = resident blocks x passes per block x warp-edges per pass
    int &S = ctx->hetn_S, &grid = ctx->hetn_grid; // decision cached per (batch size, table size)
    if (ctx->hetn_key_groups != n_groups || ctx->hetn_key_total != ctx->ht.total) {
        double best = 1e300;
        for (int s = 1; s <= WY; ++s) {
            if (WY % s) continue;
            if (s > 1 && n_b / s < 8) break;
            if (smem_of(s) > 227 * 1024) continue;
            int bps = 0;
            CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, k_het_standin<NM, NC>, 32 * WY, smem_of(s)));
            bps = std::max(1, bps);
            const int G = WY / s;
            const long long passes = ceil_div(n_groups, G);
            const int gr = (int)std::min<long long>(passes, (long long)ctx->sm_count * bps);
            const double work = (double)ceil_div(gr, ctx->sm_count) * (double)ceil_div(passes, gr) * WY * (ceil_div(n_b, s) + 1.0);
            if (work < best * 0.999) { best = work; S = s; grid = gr; }
        }
        if (best == 1e300) { S = WY; grid = (int)std::min<long long>(n_groups, ctx->sm_count); }
        ctx->hetn_key_groups = n_groups;
        ctx->hetn_key_total = ctx->ht.total;
    }
    const size_t smem = smem_of(S);
    const int P = 5 + 2 * NC * ctx->n_m;
    ProfScope prof(ctx, st);
    k_het_standin<NM, NC><<<grid, dim3(32, WY), smem, st>>>(ctx->ht, ctx->si, params, P, (int)n_w, n_groups, S,
                                                              ctx->dd.as<double>(), logL, d_h, h_h);
    LAUNCHED(ctx);
    return LL_OK;
}

template <int NC>
int launch_het_standin_modes(ll_ctx *ctx, int64_t n_w, const double *params, double *logL, double *d_h, double *h_h,
                             cudaStream_t st)
{
    switch (ctx->n_m) {
    case 1:
        if (ctx->ht1.base) return launch_het_standin1<NC>(ctx, n_w, params, logL, d_h, h_h, st);
        return launch_het_standin<1, NC>(ctx, n_w, params, logL, d_h, h_h, st);
    case 2: return launch_het_standin<2, NC>(ctx, n_w, params, logL, d_h, h_h, st);
    case 3: return launch_het_standin<3, NC>(ctx, n_w, params, logL, d_h, h_h, st);
    case 4: return launch_het_standin<4, NC>(ctx, n_w, params, logL, d_h, h_h, st);
    case 5: return launch_het_standin<5, NC>(ctx, n_w, params, logL, d_h, h_h, st);
    case 6: return launch_het_standin<6, NC>(ctx, n_w, params, logL, d_h, h_h, st);
    case 7: return launch_het_standin<7, NC>(ctx, n_w, params, logL, d_h, h_h, st);
    case 8: return launch_het_standin<8, NC>(ctx, n_w, params, logL, d_h, h_h, st);
    default: return ctx->fail(LL_ERR_UNSUPPORTED, "n_modes");
    }
}

// the heterodyned loop as ONE cooperative launch (k_pt_run_het1): single mode with the edge-regrouped table, up to 32
// temperatures.  Returns LL_ERR_UNSUPPORTED when the population or the device does not fit (the caller falls back).
template <int NC>
int pt_run_fused(ll_ctx *ctx, int32_t n_t, int32_t n_w, double *x, double *logL, double *d_h, double *h_h, const double *betas,
                 const double *lo, const double *hi, int32_t n_dim, double a, uint64_t seed, int64_t iter0, int64_t n_iter,
                 uint64_t *n_accepted, cudaStream_t st)
{
    constexpr int WY = LL_PT_WY;
    if (ctx->coop < 0) {
        int v = 0;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrCooperativeLaunch, ctx->device) != cudaSuccess) v = 0;
        ctx->coop = v;
    }
    if (!ctx->coop) return LL_ERR_UNSUPPORTED;
    const size_t tab_d = (size_t)ctx->ht1.n_e * het1_stride(NC);
    const size_t smem = sizeof(double) * (tab_d + (tab_d & 1) + (size_t)WY * 32 * 3 * NC + 7 * 32 + (size_t)WY * (32 * (5 + 2 * NC) + 16));
    if (smem > 227 * 1024) return LL_ERR_UNSUPPORTED;
    if (!ctx->ptrun_attr) {
        CK(cudaFuncSetAttribute(k_pt_run_het1<NC>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        ctx->ptrun_attr = true;
    }
    int bps = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, k_pt_run_het1<NC>, 32 * WY, smem));
    if (bps < 1) return LL_ERR_UNSUPPORTED;
    const int n_pass = ceil_div((long long)n_t * (n_w / 2), 32);
    const int grid = std::max(1, std::min(std::max(n_pass, ceil_div(n_w, WY)), ctx->sm_count * bps));
    PtRunArgs pa;
    pa.x = x; pa.logL = logL; pa.d_h = d_h; pa.h_h = h_h; pa.betas = betas; pa.lo = lo; pa.hi = hi;
    pa.dd = ctx->dd.as<double>(); pa.n_acc = (unsigned long long *)n_accepted; pa.seed = seed; pa.iter0 = iter0;
    pa.n_iter = n_iter; pa.n_t = n_t; pa.n_w = n_w; pa.n_dim = n_dim; pa.a = a;
    Het1Table tab = ctx->ht1;
    StandinInfo si = ctx->si;
    void *args[] = {&tab, &si, &pa};
    CK(cudaLaunchCooperativeKernel((const void *)k_pt_run_het1<NC>, dim3(grid), dim3(32, WY), args, smem, st));
    LAUNCHED(ctx);
    return LL_OK;
}

} // namespace

// =====================================================================================================
// C ABI
// =====================================================================================================
extern "C" {

int ll_abi_version(void) { return 3; } // 3: n_channels 2 or 3 and ll_set_data w_shared (per-channel weights), t_shift on the array
                                       // entry points, ll_standin_split_tc, ll_pt_fused

int ll_create(const ll_config *cfg, ll_ctx **out)
{
    if (!cfg || !out) return LL_ERR_ARG;
    *out = nullptr;
    if (cfg->n_channels != 2 && cfg->n_channels != 3) return LL_ERR_UNSUPPORTED;
    if (cfg->n_modes < 1 || cfg->n_modes > LL_MAX_MODES) return LL_ERR_UNSUPPORTED;
    if (cfg->precision != LL_PREC_FP64 && cfg->precision != LL_PREC_FP32_ACC) return LL_ERR_UNSUPPORTED;
    if (cfg->spline_bc != LL_BC_NATURAL && cfg->spline_bc != LL_BC_NOT_A_KNOT) return LL_ERR_UNSUPPORTED;
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || cfg->device < 0 || cfg->device >= n_dev) {
        (void)cudaGetLastError();
        return LL_ERR_CUDA; // no CUDA device: there is no CPU fallback
    }
    ll_ctx *ctx = new (std::nothrow) ll_ctx();
    if (!ctx) return LL_ERR_NOMEM;
    ctx->device = cfg->device;
    ctx->n_c = cfg->n_channels;
    ctx->n_m = cfg->n_modes;
    ctx->precision = cfg->precision;
    ctx->spline_bc = cfg->spline_bc;
    DeviceGuard dg(ctx->device);
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, ctx->device) != cudaSuccess) {
        delete ctx;
        return LL_ERR_CUDA;
    }
    if (prop.major < 10) { // the only SASS in this library is sm_100a
        delete ctx;
        return LL_ERR_UNSUPPORTED;
    }
    ctx->sm_count = prop.multiProcessorCount;
    // set-up for ll_pt_stretch_half_het_static: where this device keeps the static scratch array
    if (static_scratch_addr(ctx->device, &ctx->static_scratch) != cudaSuccess) {
        (void)cudaGetLastError();
        delete ctx;
        return LL_ERR_CUDA;
    }
    // default stand-in description: the (2,2) mode only, kappa = 1/2; overwritten by ll_standin_config
    ctx->si.n_m = ctx->n_m;
    ctx->si.kappa = 0.5;
    ctx->si.n_c = ctx->n_c;
    ctx->si.split_tc = 0;
    *out = ctx;
    return LL_OK;
}

int ll_destroy(ll_ctx *ctx)
{
    if (!ctx) return LL_ERR_ARG;
    {
        DeviceGuard dg(ctx->device);
        cudaDeviceSynchronize();
        for (auto &nb : ctx->buffers()) nb.second->release();
        for (auto &e : ctx->ev) cudaEventDestroy(e);
    }
    delete ctx;
    return LL_OK;
}

const char *ll_last_error(const ll_ctx *ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int ll_debug_check(ll_ctx *ctx, int32_t *n_bad)
{
    if (!ctx) return LL_ERR_ARG;
    DeviceGuard dg(ctx->device);
    CK(cudaDeviceSynchronize());
    int bad = 0;
    std::string names;
    for (auto &nb : ctx->buffers()) {
        const int st = nb.second->guard_state();
        if (st < 0) return ctx->fail(LL_ERR_CUDA, "guard band read-back failed");
        if (st > 0) { ++bad; names += std::string(names.empty() ? "" : ", ") + nb.first; }
    }
    if (n_bad) *n_bad = bad;
    if (bad) ctx->err = "guard band written behind: " + names;
    return LL_OK;
}

int64_t ll_kernel_launches(const ll_ctx *ctx) { return ctx ? ctx->launches : 0; }

int ll_set_data(ll_ctx *ctx, int64_t n_f, int64_t k_min, double df, const double *d, const double *W, int32_t w_shared,
                void *stream)
{
    if (!ctx) return LL_ERR_ARG;
    if (!d || !W) return ctx->fail(LL_ERR_ARG, "d or W is NULL");
    if (n_f < 1 || n_f > (1LL << 30)) return ctx->fail(LL_ERR_ARG, "n_f out of range [1, 2^30]");
    if (k_min < 0 || !(df > 0.0) || !std::isfinite(df)) return ctx->fail(LL_ERR_ARG, "k_min < 0 or df not positive");
    if (k_min + n_f >= (1LL << 31)) return ctx->fail(LL_ERR_ARG, "k_min + n_f must stay below 2^31 (bin numbers are int32 on the device)");
    if (ctx->precision == LL_PREC_FP32_ACC && (ctx->n_c != 2 || !w_shared))
        return ctx->fail(LL_ERR_UNSUPPORTED, "the FP32-accumulate variant is built for two channels sharing one weight row");
    DeviceGuard dg(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    ctx->have_data = false;
    ctx->have_het = false;
    ctx->nodes_valid = false;
    ctx->data_version += 1; // the cached frequency-tile tables and the bin -> interval table belong to the old grid
    // weight rows kept: one for two channels sharing their PSD; otherwise one per channel (a shared row is replicated)
    const int w_rows_in = w_shared ? 1 : ctx->n_c;
    const int nw = (ctx->n_c == 2 && w_shared) ? 1 : ctx->n_c;
    ctx->w_rows = nw;
    const long long n_pad = round_up(n_f, 512) + 512; // a stage of up to 512 bins may start at the grid's last bin
    CK(ctx->g.ensure(sizeof(double) * 2 * ctx->n_c * n_pad));
    CK(ctx->Wc.ensure(sizeof(double) * nw * n_pad));
    CK(ctx->dd.ensure(sizeof(double) * 2));
    const int nb = std::min(1024, ceil_div(n_f, 256));
    CK(ctx->dd_part.ensure(sizeof(double) * 1024));
    CK(cudaMemsetAsync(ctx->g.as<double>() + 2 * ctx->n_c * n_f, 0, sizeof(double) * 2 * ctx->n_c * (n_pad - n_f), st));
    for (int r = 0; r < nw; ++r)
        CK(cudaMemsetAsync(ctx->Wc.as<double>() + (size_t)r * n_pad + n_f, 0, sizeof(double) * (n_pad - n_f), st));
    CK(cudaMemsetAsync(ctx->dd.p, 0, sizeof(double) * 2, st));
#define LL_PREWEIGHT(NC) \
    k_preweight<NC><<<nb, 256, 0, st>>>(d, W, w_rows_in, nw, n_f, n_pad, ctx->g.as<double>(), ctx->Wc.as<double>(), ctx->dd_part.as<double>())
    LL_CHANNELS(ctx, LL_PREWEIGHT);
#undef LL_PREWEIGHT
    LAUNCHED(ctx);
    k_sum_parts<<<1, 256, 0, st>>>(ctx->dd_part.as<double>(), nb, ctx->dd.as<double>());
    LAUNCHED(ctx);
    if (ctx->precision == LL_PREC_FP32_ACC) {
        CK(ctx->g4f.ensure(sizeof(float) * 4 * n_pad));
        CK(ctx->Wf.ensure(sizeof(double) * n_pad));
        CK(ctx->scale.ensure(sizeof(double) * 4));
        CK(ctx->wmax.ensure(sizeof(unsigned long long)));
        CK(cudaMemsetAsync(ctx->wmax.p, 0, sizeof(unsigned long long), st));
        k_wmax<<<nb, 256, 0, st>>>(W, n_f, ctx->wmax.as<unsigned long long>());
        LAUNCHED(ctx);
        k_scale_from_wmax<<<1, 1, 0, st>>>(ctx->wmax.as<unsigned long long>(), ctx->scale.as<double>());
        LAUNCHED(ctx);
        k_prescale_f32<<<ceil_div(n_pad, 256), 256, 0, st>>>(ctx->g.as<double>(), ctx->Wc.as<double>(), n_pad,
                                                             ctx->scale.as<double>(), ctx->g4f.as<float>(), ctx->Wf.as<double>());
        LAUNCHED(ctx);
    }
    ctx->n_f = n_f;
    ctx->n_f_pad = n_pad;
    ctx->k_min = k_min;
    ctx->df = df;
    ctx->have_data = true;
    return LL_OK;
}

int ll_get_dd(ll_ctx *ctx, double *dd_full, double *dd_het_band, void *stream)
{
    if (!ctx) return LL_ERR_ARG;
    if (!ctx->have_data) return ctx->fail(LL_ERR_STATE, "ll_set_data has not been called");
    DeviceGuard dg(ctx->device);
    double h[2];
    CK(cudaMemcpyAsync(h, ctx->dd.p, sizeof(h), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    CK(cudaStreamSynchronize((cudaStream_t)stream));
    if (dd_full) *dd_full = h[0];
    if (dd_het_band) *dd_het_band = h[1];
    return LL_OK;
}

int ll_standin_config(ll_ctx *ctx, int32_t n_modes, const int32_t *l, const int32_t *m, const double *c_lm, double taper_kappa)
{
    if (!ctx) return LL_ERR_ARG;
    if (!l || !m || !c_lm) return ctx->fail(LL_ERR_ARG, "l, m or c_lm is NULL");
    if (n_modes != ctx->n_m) return ctx->fail(LL_ERR_ARG, "n_modes differs from the context's");
    if (!(taper_kappa > 0.0) || !std::isfinite(taper_kappa)) return ctx->fail(LL_ERR_ARG, "taper_kappa must be positive");
    int m_max = 0;
    for (int i = 0; i < n_modes; ++i) {
        if (m[i] < 1 || l[i] < m[i]) return ctx->fail(LL_ERR_ARG, "need 1 <= m <= l");
        m_max = std::max(m_max, (int)m[i]);
    }
    ctx->si.n_m = n_modes;
    ctx->si.m_max = m_max;
    ctx->si.kappa = taper_kappa;
    ctx->si.n_c = ctx->n_c;
    for (int i = 0; i < kMaxModes; ++i) {
        ctx->si.mode_m[i] = i < n_modes ? m[i] : 2;
        ctx->mode_l[i] = i < n_modes ? l[i] : 2;
        ctx->c_lm[i] = i < n_modes ? c_lm[i] : 0.0;
    }
    ctx->have_standin = true;
    ctx->nodes_valid = false; // node tables carry c_lm and m
    ctx->have_het = false;
    return LL_OK;
}

int ll_standin_split_tc(ll_ctx *ctx, int32_t on)
{
    if (!ctx) return LL_ERR_ARG;
    ctx->si.split_tc = on ? 1 : 0;
    return LL_OK;
}

int ll_full_batch(ll_ctx *ctx, int64_t n_w, int32_t n_nodes, const double *f_nodes, const double *amp, const double *phase,
                  const double *tf, const double *band, const double *t_shift, double *logL, double *d_h, double *h_h,
                  void *stream)
{
    int rc = check_full_common(ctx, n_w, f_nodes, logL);
    if (rc != LL_OK) return rc;
    if (n_w > 0 && (!amp || !phase || !tf)) return ctx->fail(LL_ERR_ARG, "amp, phase or tf is NULL");
    DeviceGuard dg(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    rc = prepare_nodes(ctx, n_nodes, f_nodes, st);
    if (rc != LL_OK) return rc;
    if (n_w == 0) return LL_OK;
    return run_full(ctx, n_w, n_nodes, nullptr, amp, phase, tf, band, t_shift, logL, d_h, h_h, st, false, nullptr);
}

int ll_full_batch_pw(ll_ctx *ctx, int64_t n_w, int32_t n_nodes, const double *f_nodes_w, const double *amp,
                     const double *phase, const double *tf, const double *band, const double *t_shift, double *logL,
                     double *d_h, double *h_h, void *stream)
{
    if (!ctx) return LL_ERR_ARG;
    if (n_w < 0) return ctx->fail(LL_ERR_ARG, "n_w < 0");
    if (n_w > (1 << 24)) return ctx->fail(LL_ERR_ARG, "n_w > 2^24 per call: split the batch");
    if (n_nodes < 3 || n_nodes > (1 << 20)) return ctx->fail(LL_ERR_ARG, "n_nodes out of range [3, 2^20]");
    if (n_nodes < 4 && ctx->spline_bc == LL_BC_NOT_A_KNOT) return ctx->fail(LL_ERR_ARG, "the not-a-knot boundary condition needs n_nodes >= 4");
    if (n_w > 0 && (!f_nodes_w || !amp || !phase || !tf || !logL)) return ctx->fail(LL_ERR_ARG, "NULL argument");
    if (!ctx->have_data) return ctx->fail(LL_ERR_STATE, "ll_set_data has not been called");
    if (ctx->precision != LL_PREC_FP64) return ctx->fail(LL_ERR_UNSUPPORTED, "ll_full_batch_pw is FP64 only");
    if (n_w == 0) return LL_OK;
    DeviceGuard dg(ctx->device);
    return run_full_pw(ctx, n_w, n_nodes, f_nodes_w, amp, phase, tf, band, t_shift, logL, d_h, h_h, (cudaStream_t)stream);
}

int ll_full_batch_tf(ll_ctx *ctx, int64_t n_w, int32_t n_nodes, const double *f_nodes, const double *amp,
                     const double *phase, const double *tf_nodes, const double *band, const double *t_shift, double *logL,
                     double *d_h, double *h_h, void *stream)
{
    int rc = check_full_common(ctx, n_w, f_nodes, logL);
    if (rc != LL_OK) return rc;
    if (ctx->precision != LL_PREC_FP64) return ctx->fail(LL_ERR_UNSUPPORTED, "ll_full_batch_tf is FP64 only");
    if (n_w > 0 && (!amp || !phase || !tf_nodes)) return ctx->fail(LL_ERR_ARG, "amp, phase or tf_nodes is NULL");
    DeviceGuard dg(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    rc = prepare_nodes(ctx, n_nodes, f_nodes, st);
    if (rc != LL_OK) return rc;
    if (n_w == 0) return LL_OK;
    return run_full(ctx, n_w, n_nodes, nullptr, amp, phase, nullptr, band, t_shift, logL, d_h, h_h, st, false, nullptr, tf_nodes);
}

int ll_standin_nodes(ll_ctx *ctx, int64_t n_w, int32_t n_nodes, const double *f_nodes, const double *params,
                     double *amp, double *phase, double *band, void *stream)
{
    if (!ctx) return LL_ERR_ARG;
    if (n_w < 0 || n_w > (1LL << 30)) return ctx->fail(LL_ERR_ARG, "n_w out of range");
    if (!f_nodes) return ctx->fail(LL_ERR_ARG, "f_nodes is NULL");
    if (n_w > 0 && (!params || !amp || !phase)) return ctx->fail(LL_ERR_ARG, "params, amp or phase is NULL");
    if (!ctx->have_standin) return ctx->fail(LL_ERR_STATE, "ll_standin_config has not been called");
    if (!ctx->have_data) return ctx->fail(LL_ERR_STATE, "ll_set_data has not been called (the node tables are tied to the grid)");
    DeviceGuard dg(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    int rc = prepare_nodes(ctx, n_nodes, f_nodes, st);
    if (rc != LL_OK) return rc;
    if (n_w == 0) return LL_OK;
    k_standin_nodes_out<<<(unsigned)n_w, 128, 0, st>>>(params, 5 + 2 * ctx->n_c * ctx->n_m, n_nodes, ctx->si, ctx->nt,
                                                        GridInfo{ctx->k_min, ctx->n_f, ctx->df}, amp, phase, band);
    LAUNCHED(ctx);
    return LL_OK;
}

int ll_tlm_nodes(ll_ctx *ctx, int64_t n_w, int32_t n_nodes, const double *f_nodes, const double *phase, double t_ref,
                 double *t_lm, void *stream)
{
    if (!ctx) return LL_ERR_ARG;
    if (n_w < 0) return ctx->fail(LL_ERR_ARG, "n_w < 0");
    if (!f_nodes) return ctx->fail(LL_ERR_ARG, "f_nodes is NULL");
    if (n_w > 0 && (!phase || !t_lm)) return ctx->fail(LL_ERR_ARG, "phase or t_lm is NULL");
    if (!ctx->have_data) return ctx->fail(LL_ERR_STATE, "ll_set_data has not been called (the node tables are tied to the grid)");
    if (ctx->spline_bc != LL_BC_NATURAL) return ctx->fail(LL_ERR_UNSUPPORTED, "ll_tlm_nodes differentiates the natural spline only");
    DeviceGuard dg(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    int rc = prepare_nodes(ctx, n_nodes, f_nodes, st);
    if (rc != LL_OK) return rc;
    if (n_w == 0) return LL_OK;
    const long long n_sys = n_w * ctx->n_m;
    if (n_sys > (1LL << 30)) return ctx->fail(LL_ERR_ARG, "n_w x n_modes too large");
    CK(ctx->Y.ensure(sizeof(double) * (size_t)n_sys * n_nodes));
    k_tlm_nodes<<<ceil_div(n_sys, 128), 128, 0, st>>>(phase, (int)n_sys, n_nodes, t_ref, ctx->nt, ctx->Y.as<double>(), t_lm);
    LAUNCHED(ctx);
    return LL_OK;
}

int ll_full_batch_standin(ll_ctx *ctx, int64_t n_w, int32_t n_nodes, const double *f_nodes, const double *params,
                          double *logL, double *d_h, double *h_h, void *stream)
{
    int rc = check_full_common(ctx, n_w, f_nodes, logL);
    if (rc != LL_OK) return rc;
    if (!ctx->have_standin) return ctx->fail(LL_ERR_STATE, "ll_standin_config has not been called");
    if (n_w > 0 && !params) return ctx->fail(LL_ERR_ARG, "params is NULL");
    DeviceGuard dg(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    rc = prepare_nodes(ctx, n_nodes, f_nodes, st);
    if (rc != LL_OK) return rc;
    if (n_w == 0) return LL_OK;
    return run_full(ctx, n_w, n_nodes, params, nullptr, nullptr, nullptr, nullptr, nullptr, logL, d_h, h_h, st, false, nullptr);
}

int ll_full_batch_standin_host(ll_ctx *ctx, int64_t n_w, int32_t n_nodes, const double *f_nodes, const double *params_host,
                               double *logL_host, double *d_h_host, double *h_h_host, void *stream)
{
    int rc = check_full_common(ctx, n_w, f_nodes, logL_host);
    if (rc != LL_OK) return rc;
    if (n_w == 0) return ll_full_batch_standin(ctx, 0, n_nodes, f_nodes, params_host, logL_host, d_h_host, h_h_host, stream);
    if (!params_host) return ctx->fail(LL_ERR_ARG, "params_host is NULL");
    DeviceGuard dg(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    const size_t P = 5 + 2 * (size_t)ctx->n_c * (size_t)ctx->n_m;
    CK(ctx->stage_in.ensure(sizeof(double) * P * n_w));
    CK(ctx->stage_out.ensure(sizeof(double) * 3 * n_w));
    CK(cudaMemcpyAsync(ctx->stage_in.p, params_host, sizeof(double) * P * n_w, cudaMemcpyHostToDevice, st));
    double *o = ctx->stage_out.as<double>();
    rc = ll_full_batch_standin(ctx, n_w, n_nodes, f_nodes, ctx->stage_in.as<double>(), o, o + n_w, o + 2 * n_w, stream);
    if (rc != LL_OK) return rc;
    CK(cudaMemcpyAsync(logL_host, o, sizeof(double) * n_w, cudaMemcpyDeviceToHost, st));
    if (d_h_host) CK(cudaMemcpyAsync(d_h_host, o + n_w, sizeof(double) * n_w, cudaMemcpyDeviceToHost, st));
    if (h_h_host) CK(cudaMemcpyAsync(h_h_host, o + 2 * n_w, sizeof(double) * n_w, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return LL_OK;
}

int ll_full_template_standin(ll_ctx *ctx, int32_t n_nodes, const double *f_nodes, const double *params_row, double *h_out,
                             void *stream)
{
    if (!ctx) return LL_ERR_ARG;
    if (!f_nodes || !params_row || !h_out) return ctx->fail(LL_ERR_ARG, "NULL argument");
    if (!ctx->have_data) return ctx->fail(LL_ERR_STATE, "ll_set_data has not been called (it fixes the dense grid)");
    if (!ctx->have_standin) return ctx->fail(LL_ERR_STATE, "ll_standin_config has not been called");
    DeviceGuard dg(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    int rc = prepare_nodes(ctx, n_nodes, f_nodes, st);
    if (rc != LL_OK) return rc;
    const size_t P = 5 + 2 * (size_t)ctx->n_c * (size_t)ctx->n_m;
    CK(ctx->prow.ensure(sizeof(double) * P));
    CK(cudaMemcpyAsync(ctx->prow.p, params_row, sizeof(double) * P, cudaMemcpyHostToDevice, st));
    CK(cudaStreamSynchronize(st)); // params_row is pageable caller memory
    return run_full(ctx, 1, n_nodes, ctx->prow.as<double>(), nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr,
                    nullptr, st, true, h_out);
}

int ll_template_standin(ll_ctx *ctx, const double *params_row, int64_t n_freq, const double *f, double f_lo, double f_hi,
                        double *h_out, void *stream)
{
    if (!ctx) return LL_ERR_ARG;
    if (!params_row || (n_freq > 0 && (!f || !h_out))) return ctx->fail(LL_ERR_ARG, "NULL argument");
    if (n_freq < 0) return ctx->fail(LL_ERR_ARG, "n_freq < 0");
    if (!ctx->have_standin) return ctx->fail(LL_ERR_STATE, "ll_standin_config has not been called");
    if (n_freq == 0) return LL_OK;
    DeviceGuard dg(ctx->device);
    DirectRow row;
    memset(&row, 0, sizeof(row));
    const int P = 5 + 2 * ctx->n_c * ctx->n_m;
    memcpy(row.p, params_row, sizeof(double) * P);
    memcpy(row.c_lm, ctx->c_lm, sizeof(row.c_lm));
    k_template_direct<<<ceil_div(n_freq, 256), 256, 0, (cudaStream_t)stream>>>(row, ctx->si, n_freq, f, GridInfo{0, 0, 0.0},
                                                                                f_lo, f_hi, h_out);
    LAUNCHED(ctx);
    return LL_OK;
}

int ll_het_prepare(ll_ctx *ctx, int32_t n_edges, const double *f_edges, const double *h0_dense, const double *h0_edges,
                   void *stream)
{
    if (!ctx) return LL_ERR_ARG;
    if (!f_edges || !h0_dense || !h0_edges) return ctx->fail(LL_ERR_ARG, "NULL argument");
    if (n_edges < 2 || n_edges > 65536) return ctx->fail(LL_ERR_ARG, "n_edges out of range [2, 65536]");
    for (int j = 0; j + 1 < n_edges; ++j)
        if (!(f_edges[j + 1] > f_edges[j])) return ctx->fail(LL_ERR_ARG, "f_edges must be strictly ascending and finite");
    if (!ctx->have_data) return ctx->fail(LL_ERR_STATE, "ll_set_data has not been called");
    DeviceGuard dg(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    ctx->have_het = false;
    const int n_e = n_edges, n_b = n_e - 1;
    // bin membership [e_b, e_{b+1}), last bin closed (reading R13), with the grid's own frequencies
    std::vector<int> es(n_e);
    std::vector<double> fb(n_b);
    for (int b = 0; b < n_b; ++b) {
        es[b] = (int)first_bin_ge(f_edges[b], ctx->k_min, ctx->n_f, ctx->df);
        fb[b] = (double)(0.5L * ((long double)f_edges[b] + (long double)f_edges[b + 1]));
    }
    es[n_b] = (int)first_bin_gt(f_edges[n_b], ctx->k_min, ctx->n_f, ctx->df);
    CK(ctx->het_idx.ensure(sizeof(int) * n_e));
    CK(ctx->het_fb.ensure(sizeof(double) * n_b));
    const int NR = 6 * ctx->n_c + 1; // raw sums per bin: per channel (A0r, A0i, A1r, A1i, B0, B1), then <d|d>
    CK(ctx->het_raw.ensure(sizeof(double) * NR * n_b));
    CK(cudaMemcpyAsync(ctx->het_idx.p, es.data(), sizeof(int) * n_e, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(ctx->het_fb.p, fb.data(), sizeof(double) * n_b, cudaMemcpyHostToDevice, st));
    const GridInfo g{ctx->k_min, ctx->n_f, ctx->df};
#define LL_HETPREP(NC)                                                                                                 \
    k_het_prepare<NC><<<n_b, 256, 0, st>>>(ctx->g.as<double>(), ctx->Wc.as<double>(), ctx->w_rows, ctx->n_f_pad, h0_dense, g, \
                                           ctx->het_idx.as<int>(), ctx->het_fb.as<double>(), ctx->het_raw.as<double>())
    LL_CHANNELS(ctx, LL_HETPREP);
#undef LL_HETPREP
    LAUNCHED(ctx);
    ctx->raw_host.assign((size_t)NR * n_b, 0.0);
    std::vector<double> h0e((size_t)ctx->n_c * n_e * 2);
    CK(cudaMemcpyAsync(ctx->raw_host.data(), ctx->het_raw.p, sizeof(double) * NR * n_b, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(h0e.data(), h0_edges, sizeof(double) * h0e.size(), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    std::vector<double> tab;
    int rc = build_het_table(ctx, n_e, f_edges, h0e, tab);
    if (rc != LL_OK) return rc;
    // <d|d> over the band: bins in a fixed order, compensated
    long double ddb = 0.0L;
    for (int b = 0; b < n_b; ++b) ddb += (long double)ctx->raw_host[(size_t)b * NR + NR - 1];
    const double ddb_d = (double)ddb;
    CK(ctx->het_tab.ensure(sizeof(double) * tab.size()));
    CK(cudaMemcpyAsync(ctx->het_tab.p, tab.data(), sizeof(double) * tab.size(), cudaMemcpyHostToDevice, st));
    std::vector<double> tab1;
    ctx->ht1 = Het1Table{nullptr, n_e, n_b};
    if (ctx->n_m == 1 && ctx->have_standin) {
        build_het1_table(ctx, n_e, f_edges, h0e, tab1);
        CK(ctx->het_tab1.ensure(sizeof(double) * tab1.size()));
        CK(cudaMemcpyAsync(ctx->het_tab1.p, tab1.data(), sizeof(double) * tab1.size(), cudaMemcpyHostToDevice, st));
        ctx->ht1.base = ctx->het_tab1.as<double>();
    }
    CK(cudaMemcpyAsync(ctx->dd.as<double>() + 1, &ddb_d, sizeof(double), cudaMemcpyHostToDevice, st));
    CK(cudaStreamSynchronize(st));
    ctx->ht.base = ctx->het_tab.as<double>();
    ctx->n_e = n_e;
    ctx->have_het = true;
    return LL_OK;
}

// H0 inside the sampling loop: the highest-likelihood walker becomes the reference; the band is where
// h0 != 0 (reading R12: log-spaced edges from the grid's first frequency to min(f_last, f_ISCO)).
int ll_het_refresh_standin(ll_ctx *ctx, int64_t n_w, const double *params, const double *logL, int32_t n_edges,
                           int64_t *best_index, double *f_edges_out, void *stream)
{
    if (!ctx) return LL_ERR_ARG;
    if (n_w <= 0 || n_w > (1LL << 30)) return ctx->fail(LL_ERR_ARG, "n_w out of range (needs at least one walker)");
    if (!params || !logL) return ctx->fail(LL_ERR_ARG, "params or logL is NULL");
    if (n_edges < 2 || n_edges > 65536) return ctx->fail(LL_ERR_ARG, "n_edges out of range [2, 65536]");
    if (!ctx->have_data) return ctx->fail(LL_ERR_STATE, "ll_set_data has not been called");
    if (!ctx->have_standin) return ctx->fail(LL_ERR_STATE, "ll_standin_config has not been called");
    DeviceGuard dg(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    const int P = 5 + 2 * ctx->n_c * ctx->n_m;
    CK(ctx->ref_idx.ensure(sizeof(long long)));
    k_argmax<<<1, 1024, 0, st>>>(logL, (long long)n_w, ctx->ref_idx.as<long long>());
    LAUNCHED(ctx);
    long long best = -1;
    CK(cudaMemcpyAsync(&best, ctx->ref_idx.p, sizeof(long long), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (best < 0) return ctx->fail(LL_ERR_ARG, "no finite log L in the population");
    DirectRow row;
    memset(&row, 0, sizeof(row));
    CK(cudaMemcpyAsync(row.p, params + (size_t)best * P, sizeof(double) * P, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    memcpy(row.c_lm, ctx->c_lm, sizeof(row.c_lm));
    // edges: geomspace(f_0, min(f_last, f_ISCO(best)), n_edges), end points exact
    const double q = row.p[1];
    const double eta = q / ((1.0 + q) * (1.0 + q));
    const double f_isco = 0x1.16b28f55d72d4p-4 / (3.14159265358979323846 * row.p[0] * std::pow(eta, -0.6));
    const double f_first = bin_freq(ctx->k_min, 0, ctx->df), f_last = bin_freq(ctx->k_min, ctx->n_f - 1, ctx->df);
    const double f_top = std::min(f_last, f_isco);
    if (!(f_top > f_first)) return ctx->fail(LL_ERR_REF_ZERO, "the best walker's f_ISCO lies below the grid: no heterodyne band");
    std::vector<double> e((size_t)n_edges);
    const long double l0 = std::log((long double)f_first), l1 = std::log((long double)f_top);
    for (int j = 0; j < n_edges; ++j) e[j] = (double)std::exp(l0 + (l1 - l0) * (long double)j / (long double)(n_edges - 1));
    e[0] = f_first;
    e[n_edges - 1] = f_top;
    CK(ctx->ref_dense.ensure(sizeof(double) * 2 * ctx->n_c * (size_t)ctx->n_f));
    CK(ctx->ref_edges.ensure(sizeof(double) * (2 * ctx->n_c + 1) * (size_t)n_edges));
    double *fe_dev = ctx->ref_edges.as<double>() + (size_t)2 * ctx->n_c * n_edges;
    CK(cudaMemcpyAsync(fe_dev, e.data(), sizeof(double) * n_edges, cudaMemcpyHostToDevice, st));
    const GridInfo g{ctx->k_min, ctx->n_f, ctx->df};
    k_template_direct<<<ceil_div(ctx->n_f, 256), 256, 0, st>>>(row, ctx->si, ctx->n_f, nullptr, g, f_first, f_last,
                                                               ctx->ref_dense.as<double>());
    LAUNCHED(ctx);
    k_template_direct<<<ceil_div(n_edges, 256), 256, 0, st>>>(row, ctx->si, n_edges, fe_dev, g, f_first, f_last,
                                                              ctx->ref_edges.as<double>());
    LAUNCHED(ctx);
    int rc = ll_het_prepare(ctx, n_edges, e.data(), ctx->ref_dense.as<double>(), ctx->ref_edges.as<double>(), stream);
    if (rc != LL_OK) return rc;
    if (best_index) *best_index = best;
    if (f_edges_out) memcpy(f_edges_out, e.data(), sizeof(double) * n_edges);
    return LL_OK;
}

// brute-force dense log L over the heterodyne band, template evaluated directly at every dense bin
int ll_het_audit_standin(ll_ctx *ctx, int64_t n_w, const double *params, double *logL, double *d_h, double *h_h,
                         void *stream)
{
    int rc = het_check(ctx, n_w, logL);
    if (rc != LL_OK) return rc;
    if (!ctx->have_standin) return ctx->fail(LL_ERR_STATE, "ll_standin_config has not been called");
    if (n_w == 0) return LL_OK;
    if (!params) return ctx->fail(LL_ERR_ARG, "params is NULL");
    DeviceGuard dg(ctx->device);
    DirectClm cl;
    memcpy(cl.c_lm, ctx->c_lm, sizeof(cl.c_lm));
    const GridInfo g{ctx->k_min, ctx->n_f, ctx->df};
#define LL_AUDIT(NC)                                                                                                   \
    k_het_audit<NC><<<(unsigned)n_w, 256, 0, (cudaStream_t)stream>>>(params, 5 + 2 * ctx->n_c * ctx->n_m, cl, ctx->si,   \
                                                                     ctx->g.as<double>(), ctx->Wc.as<double>(), ctx->w_rows, \
                                                                     ctx->n_f_pad, g, ctx->het_idx.as<int>(), ctx->n_e - 1, \
                                                                     ctx->dd.as<double>(), logL, d_h, h_h)
    LL_CHANNELS(ctx, LL_AUDIT);
#undef LL_AUDIT
    LAUNCHED(ctx);
    return LL_OK;
}

int ll_het_get_summary(ll_ctx *ctx, double *A0, double *A1, double *B0, double *B1, void *stream)
{
    (void)stream;
    if (!ctx) return LL_ERR_ARG;
    if (!ctx->have_het) return ctx->fail(LL_ERR_STATE, "ll_het_prepare has not been called");
    const int n_b = ctx->n_e - 1, NR = 6 * ctx->n_c + 1;
    for (int c = 0; c < ctx->n_c; ++c)
        for (int b = 0; b < n_b; ++b) {
            const double *r = &ctx->raw_host[(size_t)b * NR + 6 * c];
            if (A0) { A0[((size_t)c * n_b + b) * 2] = r[0]; A0[((size_t)c * n_b + b) * 2 + 1] = r[1]; }
            if (A1) { A1[((size_t)c * n_b + b) * 2] = r[2]; A1[((size_t)c * n_b + b) * 2 + 1] = r[3]; }
            if (B0) B0[(size_t)c * n_b + b] = r[4];
            if (B1) B1[(size_t)c * n_b + b] = r[5];
        }
    return LL_OK;
}

int ll_het_batch(ll_ctx *ctx, int64_t n_w, const double *amp_e, const double *phase_e, const double *tf, const double *t_shift,
                 double *logL, double *d_h, double *h_h, void *stream)
{
    int rc = het_check(ctx, n_w, logL);
    if (rc != LL_OK) return rc;
    if (n_w == 0) return LL_OK;
    if (!amp_e || !phase_e || !tf) return ctx->fail(LL_ERR_ARG, "amp_e, phase_e or tf is NULL");
    DeviceGuard dg(ctx->device);
    const size_t smem = sizeof(double) * (size_t)ctx->ht.total;
    if (smem > 227 * 1024) return ctx->fail(LL_ERR_UNSUPPORTED, "heterodyne tables exceed shared memory");
    if (!ctx->heta_attr) {
#define LL_HETA_ATTR(NC) CK(cudaFuncSetAttribute(k_het_arrays<NC>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024))
        LL_CHANNELS(ctx, LL_HETA_ATTR);
#undef LL_HETA_ATTR
        ctx->heta_attr = true;
    }
    const int wpb = 8;
    int blocks_per_sm = std::max(1, std::min(8, (int)((220 * 1024) / std::max<size_t>(smem, 1))));
    const int grid = std::min(ceil_div(n_w, wpb), ctx->sm_count * blocks_per_sm);
    ProfScope prof(ctx, (cudaStream_t)stream);
#define LL_HETA(NC)                                                                                                       \
    k_het_arrays<NC><<<grid, wpb * 32, smem, (cudaStream_t)stream>>>(ctx->ht, amp_e, phase_e, tf, t_shift, (int)n_w,       \
                                                                      ctx->dd.as<double>(), logL, d_h, h_h)
    LL_CHANNELS(ctx, LL_HETA);
#undef LL_HETA
    LAUNCHED(ctx);
    return LL_OK;
}

int ll_het_batch_standin(ll_ctx *ctx, int64_t n_w, const double *params, double *logL, double *d_h, double *h_h, void *stream)
{
    int rc = het_check(ctx, n_w, logL);
    if (rc != LL_OK) return rc;
    if (!ctx->have_standin) return ctx->fail(LL_ERR_STATE, "ll_standin_config has not been called");
    if (n_w == 0) return LL_OK;
    if (!params) return ctx->fail(LL_ERR_ARG, "params is NULL");
    DeviceGuard dg(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    if (ctx->n_c == 2) return launch_het_standin_modes<2>(ctx, n_w, params, logL, d_h, h_h, st);
    return launch_het_standin_modes<3>(ctx, n_w, params, logL, d_h, h_h, st);
}

int ll_het_batch_standin_host(ll_ctx *ctx, int64_t n_w, const double *params_host, double *logL_host, double *d_h_host,
                              double *h_h_host, void *stream)
{
    int rc = het_check(ctx, n_w, logL_host);
    if (rc != LL_OK) return rc;
    if (n_w == 0) return LL_OK;
    if (!params_host) return ctx->fail(LL_ERR_ARG, "params_host is NULL");
    DeviceGuard dg(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    const size_t P = 5 + 2 * (size_t)ctx->n_c * (size_t)ctx->n_m;
    CK(ctx->stage_in.ensure(sizeof(double) * P * n_w));
    CK(ctx->stage_out.ensure(sizeof(double) * 3 * n_w));
    CK(cudaMemcpyAsync(ctx->stage_in.p, params_host, sizeof(double) * P * n_w, cudaMemcpyHostToDevice, st));
    double *o = ctx->stage_out.as<double>();
    rc = ll_het_batch_standin(ctx, n_w, ctx->stage_in.as<double>(), o, o + n_w, o + 2 * n_w, stream);
    if (rc != LL_OK) return rc;
    CK(cudaMemcpyAsync(logL_host, o, sizeof(double) * n_w, cudaMemcpyDeviceToHost, st));
    if (d_h_host) CK(cudaMemcpyAsync(d_h_host, o + n_w, sizeof(double) * n_w, cudaMemcpyDeviceToHost, st));
    if (h_h_host) CK(cudaMemcpyAsync(h_h_host, o + 2 * n_w, sizeof(double) * n_w, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return LL_OK;
}

// ---- sampler step around the likelihood (readings R25-R28) ----------------
namespace {
int pt_half(ll_ctx *ctx, bool full, int32_t n_nodes, const double *f_nodes, int32_t n_t, int32_t n_w, int32_t half,
            double *x, double *logL, double *d_h, double *h_h, const double *betas, const double *lo, const double *hi,
            int32_t n_dim, double a, const double *u_z, const double *u_partner, const double *u_accept,
            int32_t *accepted, void *stream, unsigned long long *n_acc = nullptr)
{
    if (!ctx) return LL_ERR_ARG;
    if (n_t < 1 || n_w < 2 || (n_w & 1)) return ctx->fail(LL_ERR_ARG, "n_temps >= 1 and an even n_walkers >= 2 are required");
    if ((int64_t)n_t * n_w > (1LL << 30)) return ctx->fail(LL_ERR_ARG, "n_temps * n_walkers too large");
    if (half != 0 && half != 1) return ctx->fail(LL_ERR_ARG, "half must be 0 or 1");
    if (!x || !logL || !betas || !lo || !hi || !u_z || !u_partner || !u_accept) return ctx->fail(LL_ERR_ARG, "NULL argument");
    if (n_dim < 1 || !(a > 1.0)) return ctx->fail(LL_ERR_ARG, "n_dim >= 1 and a > 1 are required");
    if (!ctx->have_standin) return ctx->fail(LL_ERR_STATE, "ll_standin_config has not been called");
    DeviceGuard dg(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    const int P = 5 + 2 * ctx->n_c * ctx->n_m;
    const int64_t np = (int64_t)n_t * (n_w / 2);
    CK(ctx->pt_y.ensure(sizeof(double) * (size_t)np * P));
    CK(ctx->pt_out.ensure(sizeof(double) * (size_t)np * 4));
    CK(ctx->pt_in.ensure(sizeof(int) * (size_t)np));
    double *y = ctx->pt_y.as<double>(), *ly = ctx->pt_out.as<double>(), *ydh = ly + np, *yhh = ly + 2 * np, *lnz = ly + 3 * np;
    const int grid = (int)ceil_div(np, 128);
    k_pt_propose<<<grid, 128, 0, st>>>(x, n_t, n_w, P, half, a, n_dim, lo, hi, u_z, u_partner, y, lnz, ctx->pt_in.as<int>());
    LAUNCHED(ctx);
    int rc = full ? ll_full_batch_standin(ctx, np, n_nodes, f_nodes, y, ly, ydh, yhh, stream)
                  : ll_het_batch_standin(ctx, np, y, ly, ydh, yhh, stream);
    if (rc != LL_OK) return rc;
    k_pt_accept<<<grid, 128, 0, st>>>(x, logL, d_h, h_h, n_t, n_w, P, half, betas, u_accept, y, ly, ydh, yhh, lnz,
                                      ctx->pt_in.as<int>(), accepted, n_acc);
    LAUNCHED(ctx);
    return LL_OK;
}
} // namespace

int ll_pt_stretch_half_het(ll_ctx *ctx, int32_t n_temps, int32_t n_walkers, int32_t half, double *x, double *logL,
                           double *d_h, double *h_h, const double *betas, const double *lo, const double *hi,
                           int32_t n_dim, double a, const double *u_z, const double *u_partner, const double *u_accept,
                           int32_t *accepted, void *stream)
{
    return pt_half(ctx, false, 0, nullptr, n_temps, n_walkers, half, x, logL, d_h, h_h, betas, lo, hi, n_dim, a, u_z,
                   u_partner, u_accept, accepted, stream);
}

// The same half update with the proposal rows, the proposals' results and the inside-the-box flags in the static
// device array instead of the context's lazily grown buffers: no cudaMalloc, cudaFree or allocating library call on
// this path (k_pt_propose, the H1-H3 kernel of ll_het_batch_standin, k_pt_accept: three launches, the same kernels and
// arithmetic as ll_pt_stretch_half_het).  Nothing in the scratch has to start at zero: k_pt_propose writes every row,
// ln z and flag of the call's proposals and the likelihood kernel every result before k_pt_accept reads them; what a
// previous call left behind is never read.
int ll_pt_stretch_half_het_static(ll_ctx *ctx, int32_t n_temps, int32_t n_walkers, int32_t half, double *x, double *logL,
                                  double *d_h, double *h_h, const double *betas, const double *lo, const double *hi,
                                  int32_t n_dim, double a, const double *u_z, const double *u_partner,
                                  const double *u_accept, int32_t *accepted, void *stream)
{
    if (!ctx) return LL_ERR_ARG;
    if (n_temps < 1 || n_walkers < 2 || (n_walkers & 1))
        return ctx->fail(LL_ERR_ARG, "n_temps >= 1 and an even n_walkers >= 2 are required");
    if (half != 0 && half != 1) return ctx->fail(LL_ERR_ARG, "half must be 0 or 1");
    if (!x || !logL || !betas || !lo || !hi || !u_z || !u_partner || !u_accept) return ctx->fail(LL_ERR_ARG, "NULL argument");
    if (n_dim < 1 || !(a > 1.0)) return ctx->fail(LL_ERR_ARG, "n_dim >= 1 and a > 1 are required");
    if (!ctx->have_standin) return ctx->fail(LL_ERR_STATE, "ll_standin_config has not been called");
    if (!ctx->static_scratch) return ctx->fail(LL_ERR_STATE, "the static scratch array has no device address (ll_create)");
    const int P = 5 + 2 * ctx->n_c * ctx->n_m;
    const int64_t np = (int64_t)n_temps * (n_walkers / 2);
    // layout in doubles: y [np][P] | ln L(y), <d|h>, <h|h>, (n_dim - 1) ln z [4][np] | flags (int) [np]
    const int64_t need = np * (P + 4) + (np + 1) / 2;
    const int64_t have = (int64_t)(LL_STATIC_SCRATCH_BYTES / sizeof(double));
    if (need > have)
        return ctx->fail(LL_ERR_ARG, "ll_pt_stretch_half_het_static: n_temps * n_walkers / 2 = " + std::to_string(np) + " proposals of " +
                                         std::to_string(P) + " parameters need " + std::to_string(need * 8) +
                                         " bytes of scratch, the static array holds LL_STATIC_SCRATCH_BYTES = " +
                                         std::to_string((long long)LL_STATIC_SCRATCH_BYTES) + " (use ll_pt_stretch_half_het)");
    DeviceGuard dg(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    double *y = ctx->static_scratch, *ly = y + np * P, *ydh = ly + np, *yhh = ly + 2 * np, *lnz = ly + 3 * np;
    int *inside = reinterpret_cast<int *>(ly + 4 * np);
    const int grid = (int)ceil_div(np, 128);
    k_pt_propose<<<grid, 128, 0, st>>>(x, n_temps, n_walkers, P, half, a, n_dim, lo, hi, u_z, u_partner, y, lnz, inside);
    LAUNCHED(ctx);
    const int rc = ll_het_batch_standin(ctx, np, y, ly, ydh, yhh, stream);
    if (rc != LL_OK) return rc;
    k_pt_accept<<<grid, 128, 0, st>>>(x, logL, d_h, h_h, n_temps, n_walkers, P, half, betas, u_accept, y, ly, ydh, yhh, lnz,
                                      inside, accepted, nullptr);
    LAUNCHED(ctx);
    return LL_OK;
}

int ll_pt_stretch_half_full(ll_ctx *ctx, int32_t n_nodes, const double *f_nodes, int32_t n_temps, int32_t n_walkers,
                            int32_t half, double *x, double *logL, double *d_h, double *h_h, const double *betas,
                            const double *lo, const double *hi, int32_t n_dim, double a, const double *u_z,
                            const double *u_partner, const double *u_accept, int32_t *accepted, void *stream)
{
    return pt_half(ctx, true, n_nodes, f_nodes, n_temps, n_walkers, half, x, logL, d_h, h_h, betas, lo, hi, n_dim, a, u_z,
                   u_partner, u_accept, accepted, stream);
}

int ll_pt_swap(ll_ctx *ctx, int32_t n_temps, int32_t n_walkers, double *x, double *logL, double *d_h, double *h_h,
               const double *betas, const double *u_swap, int32_t *swapped, void *stream)
{
    if (!ctx) return LL_ERR_ARG;
    if (n_temps < 1 || n_walkers < 1) return ctx->fail(LL_ERR_ARG, "n_temps, n_walkers >= 1 are required");
    if (!x || !logL || !betas || (n_temps > 1 && !u_swap)) return ctx->fail(LL_ERR_ARG, "NULL argument");
    if (n_temps == 1) return LL_OK;
    DeviceGuard dg(ctx->device);
    const int P = 5 + 2 * ctx->n_c * ctx->n_m;
    if (n_temps <= 32 && P <= 64)
        k_pt_swap_warp<<<(int)ceil_div(n_walkers, 4), 128, 0, (cudaStream_t)stream>>>(x, logL, d_h, h_h, n_temps, n_walkers, P,
                                                                                     betas, u_swap, swapped);
    else
        k_pt_swap<<<(int)ceil_div(n_walkers, 128), 128, 0, (cudaStream_t)stream>>>(x, logL, d_h, h_h, n_temps, n_walkers, P,
                                                                                  betas, u_swap, swapped);
    LAUNCHED(ctx);
    return LL_OK;
}

// n_iter whole iterations (half 0, half 1, swap sweep) with the library's own counter-based uniforms (reading R31):
// every launch is enqueued on `stream`, nothing returns to the host in between.
namespace {
int pt_run(ll_ctx *ctx, bool full, int32_t n_nodes, const double *f_nodes, int32_t n_t, int32_t n_w, double *x, double *logL,
           double *d_h, double *h_h, const double *betas, const double *lo, const double *hi, int32_t n_dim, double a,
           uint64_t seed, int64_t iter0, int64_t n_iter, uint64_t *n_accepted, void *stream)
{
    if (!ctx) return LL_ERR_ARG;
    if (n_iter < 0 || iter0 < 0) return ctx->fail(LL_ERR_ARG, "iter0, n_iter >= 0 are required");
    if (n_t < 1 || n_w < 2 || (n_w & 1)) return ctx->fail(LL_ERR_ARG, "n_temps >= 1 and an even n_walkers >= 2 are required");
    if ((int64_t)n_t * n_w > (1LL << 28)) return ctx->fail(LL_ERR_ARG, "n_temps * n_walkers too large");
    DeviceGuard dg(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    if (!full && ctx->pt_fused && ctx->n_m == 1 && n_t <= 32 && n_iter > 0) {
        // the same checks pt_half makes, then the whole loop in one cooperative launch
        if (!x || !logL || !betas || !lo || !hi) return ctx->fail(LL_ERR_ARG, "NULL argument");
        if (n_dim < 1 || !(a > 1.0)) return ctx->fail(LL_ERR_ARG, "n_dim >= 1 and a > 1 are required");
        int rc = het_check(ctx, (int64_t)n_t * n_w, logL);
        if (rc != LL_OK) return rc;
        if (!ctx->have_standin) return ctx->fail(LL_ERR_STATE, "ll_standin_config has not been called");
        if (ctx->ht1.base) {
            rc = ctx->n_c == 2 ? pt_run_fused<2>(ctx, n_t, n_w, x, logL, d_h, h_h, betas, lo, hi, n_dim, a, seed, iter0, n_iter, n_accepted, st)
                               : pt_run_fused<3>(ctx, n_t, n_w, x, logL, d_h, h_h, betas, lo, hi, n_dim, a, seed, iter0, n_iter, n_accepted, st);
            if (rc != LL_ERR_UNSUPPORTED) return rc;
        }
    }
    const int n_half = n_t * (n_w / 2), n_swap = (n_t - 1) * n_w;
    CK(ctx->pt_u.ensure(sizeof(double) * (size_t)(6 * n_half + n_swap)));
    double *u = ctx->pt_u.as<double>();
    for (int64_t it = iter0; it < iter0 + n_iter; ++it) {
        k_pt_uniforms<<<ceil_div(6 * n_half + n_swap, 256), 256, 0, st>>>(seed, it, n_half, n_swap, u);
        LAUNCHED(ctx);
        for (int half = 0; half < 2; ++half) {
            const double *uh = u + (size_t)3 * half * n_half;
            int rc = pt_half(ctx, full, n_nodes, f_nodes, n_t, n_w, half, x, logL, d_h, h_h, betas, lo, hi, n_dim, a, uh,
                             uh + n_half, uh + 2 * (size_t)n_half, nullptr, stream, (unsigned long long *)n_accepted);
            if (rc != LL_OK) return rc;
        }
        if (n_t > 1) {
            int rc = ll_pt_swap(ctx, n_t, n_w, x, logL, d_h, h_h, betas, u + (size_t)6 * n_half, nullptr, stream);
            if (rc != LL_OK) return rc;
        }
    }
    return LL_OK;
}
} // namespace

int ll_pt_run_het(ll_ctx *ctx, int32_t n_temps, int32_t n_walkers, double *x, double *logL, double *d_h, double *h_h,
                  const double *betas, const double *lo, const double *hi, int32_t n_dim, double a, uint64_t seed,
                  int64_t iter0, int64_t n_iter, uint64_t *n_accepted, void *stream)
{
    return pt_run(ctx, false, 0, nullptr, n_temps, n_walkers, x, logL, d_h, h_h, betas, lo, hi, n_dim, a, seed, iter0, n_iter,
                  n_accepted, stream);
}

int ll_pt_run_full(ll_ctx *ctx, int32_t n_nodes, const double *f_nodes, int32_t n_temps, int32_t n_walkers, double *x,
                   double *logL, double *d_h, double *h_h, const double *betas, const double *lo, const double *hi,
                   int32_t n_dim, double a, uint64_t seed, int64_t iter0, int64_t n_iter, uint64_t *n_accepted, void *stream)
{
    return pt_run(ctx, true, n_nodes, f_nodes, n_temps, n_walkers, x, logL, d_h, h_h, betas, lo, hi, n_dim, a, seed, iter0,
                  n_iter, n_accepted, stream);
}

int ll_pt_fused(ll_ctx *ctx, int32_t on)
{
    if (!ctx) return LL_ERR_ARG;
    ctx->pt_fused = on != 0;
    return LL_OK;
}

int ll_pt_stats(ll_ctx *ctx, int64_t n, const double *logL, const double *d_h, const double *h_h, double *out3, void *stream)
{
    if (!ctx) return LL_ERR_ARG;
    if (n < 1 || !logL || !out3) return ctx->fail(LL_ERR_ARG, "n >= 1, logL and out3 are required");
    DeviceGuard dg(ctx->device);
    k_pt_stats<<<1, 1024, 0, (cudaStream_t)stream>>>(logL, d_h, h_h, (long long)n, out3);
    LAUNCHED(ctx);
    return LL_OK;
}

int ll_stop_snr(double extracted_snr, double limit) { return extracted_snr >= limit ? 1 : 0; }

int ll_stop_converged(ll_stop_state *s, double max_logL)
{
    if (!s) return LL_ERR_ARG;
    if (!s->has_ref || !(fabs(max_logL - s->ref) < s->tol)) {
        s->ref = max_logL;
        s->count = 0;
        s->has_ref = 1;
    } else {
        s->count += 1;
    }
    return s->count >= s->n_checks ? 1 : 0;
}

int ll_peak_fma(ll_ctx *ctx, int32_t which, int64_t iters, double *fma_per_s, double *ms_out, void *stream)
{
    if (!ctx) return LL_ERR_ARG;
    if (iters < 1 || which < 0 || which > 7) return ctx->fail(LL_ERR_ARG, "bad which/iters");
    DeviceGuard dg(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    CK(ctx->prow.ensure(256));
    CK(cudaMemsetAsync(ctx->prow.p, 0, 256, st));
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    const int blocks = ctx->sm_count * 8, threads = 256;
    const int64_t iters_timed = iters;
    for (int rep = 0; rep < 2; ++rep) { // first pass warms up (a short one when the timed pass runs for seconds)
        iters = rep == 0 ? std::min<int64_t>(iters_timed, 4000) : iters_timed;
        CK(cudaEventRecord(e0, st));
        if (which == 0) k_peak_fma<double><<<blocks, threads, 0, st>>>(iters, ctx->prow.as<double>());
        else if (which == 1) k_peak_fma<float><<<blocks, threads, 0, st>>>(iters, ctx->prow.as<float>());
        else if (which == 2) k_peak_dfma_pattern<0><<<blocks, threads, 0, st>>>(iters, ctx->prow.as<double>());
        else if (which == 3) k_peak_dfma_pattern<1><<<blocks, threads, 0, st>>>(iters, ctx->prow.as<double>());
        else if (which == 4) k_peak_dfma_mix<0, 16><<<blocks, threads, 0, st>>>(iters, ctx->prow.as<double>());
        else if (which == 5) k_peak_dfma_mix<0, 32><<<blocks, threads, 0, st>>>(iters, ctx->prow.as<double>());
        else if (which == 6) k_peak_dfma_mix<1, 16><<<blocks, threads, 0, st>>>(iters, ctx->prow.as<double>());
        else k_peak_dfma_mix<1, 32><<<blocks, threads, 0, st>>>(iters, ctx->prow.as<double>());
        LAUNCHED(ctx);
        CK(cudaEventRecord(e1, st));
        CK(cudaEventSynchronize(e1));
    }
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, e0, e1));
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    const double n_fma = (double)blocks * threads * (double)iters * 32.0;
    if (fma_per_s) *fma_per_s = n_fma / (ms * 1e-3);
    if (ms_out) *ms_out = ms;
    return LL_OK;
}

int ll_profile_enable(ll_ctx *ctx, int32_t on)
{
    if (!ctx) return LL_ERR_ARG;
    DeviceGuard dg(ctx->device);
    if (on && ctx->ev.empty()) {
        ctx->ev.resize(2 * kEvPairs);
        for (auto &e : ctx->ev) CK(cudaEventCreate(&e));
    }
    ctx->profiling = on != 0;
    ctx->ev_used = 0;
    return LL_OK;
}

int ll_profile_read(ll_ctx *ctx, double *kernel_ms_sum, int64_t *n_launches)
{
    if (!ctx) return LL_ERR_ARG;
    DeviceGuard dg(ctx->device);
    double sum = 0.0;
    const int n = std::min(ctx->ev_used, kEvPairs);
    for (int i = 0; i < n; ++i) {
        float ms = 0.f;
        CK(cudaEventSynchronize(ctx->ev[2 * i + 1]));
        CK(cudaEventElapsedTime(&ms, ctx->ev[2 * i], ctx->ev[2 * i + 1]));
        sum += ms;
    }
    if (kernel_ms_sum) *kernel_ms_sum = sum;
    if (n_launches) *n_launches = n;
    return LL_OK;
}

int ll_last_full_stats(ll_ctx *ctx, double *active_pairs, int64_t *n_blocks, void *stream)
{
    if (!ctx) return LL_ERR_ARG;
    if (!ctx->pairs.p) return ctx->fail(LL_ERR_STATE, "no full-grid call yet");
    DeviceGuard dg(ctx->device);
    unsigned long long v = 0;
    CK(cudaMemcpyAsync(&v, ctx->pairs.p, sizeof(v), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    CK(cudaStreamSynchronize((cudaStream_t)stream));
    if (active_pairs) *active_pairs = (double)v;
    if (n_blocks) *n_blocks = ctx->last_n_blocks;
    return LL_OK;
}

} // extern "C"
