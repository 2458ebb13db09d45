/*
 * ll.h — C ABI of the B200-native batched LISA MBHB log-likelihood library (libll_b200.so).
 *
 * What it computes (arXiv:2111.01064, text in /root/reference/PAPER.md; readings R1..R23 in DESIGN.md §3):
 *   log L = -1/2 <d-h|d-h> = <d|h> - 1/2 <h|h> - 1/2 <d|d>                         Eq. 2
 *   <a|b> = 4 Re sum_{A,E} int a~*(f) b~(f) / S_n(f) df                            Eq. 3
 *   h~_lm(f) = A_lm(f) exp(-i phi_lm(f)),  h~^{A,E}(f) = sum_lm T^{A,E}_lm h~_lm   Eq. 7, 9
 *   heterodyne: r = h/h0 = r0 + r1 (f - f_b);  Z[d,h], Z[h,h] from A0,A1,B0,B1     Eq. 10-19
 * for a whole batch of parameter points ("walkers") per call, in two forms:
 *   full-grid    (brute-force search): sparse-node amp/phase -> natural cubic spline -> dense
 *                Fourier grid -> <d|h>, <h|h> per walker; the dense template never touches HBM.
 *   heterodyned: template at the bin edges -> r -> r0, r1 -> contraction with
 *                the summary data.
 *
 * Conventions
 *   - Every function returns an int status (LL_OK = 0, negative = error) and never throws or aborts;
 *     ll_last_error() gives the text of the last failure on that context.
 *   - Pointers are marked DEV (device memory on the context's device), HOST, or PINNED (page-locked host).
 *     The caller owns every pointer it passes.  The library copies what it keeps (pre-weighted data,
 *     weights, summary tables) and holds no caller pointer once the stream has reached the end of the call.
 *   - All arrays are row-major fp64.  Complex numbers are (re, im) pairs in the last axis.
 *   - n_c = ll_config.n_channels: 2 (TDI A, E) or 3 (A, E, T; Eq. 3 sums over all three).
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Batch calls are
 *     asynchronous on it, never synchronise, and do not allocate in steady state (scratch grows on the
 *     first call at a larger shape; growing synchronises the device once).
 *   - A context is not thread-safe: one context per host thread / stream.
 *   - Non-finite inputs propagate to NaN outputs unchecked.  A walker whose band misses the grid gets
 *     d_h = h_h = 0, log L = -1/2 <d|d>.
 *   - There is no CPU fallback anywhere: without a CUDA device ll_create fails with LL_ERR_CUDA.
 *
 * Dense grid (reading R3): bin i = 0..n_f-1 has frequency f_i = (double)(k_min + i) * df.
 * Weights (reading R4):    W_i = 4 df w_i / S_n(f_i), w_i the quadrature weight (trapezoid or rectangle).
 * Parameter row of the stand-in waveform (reading R9; BASELINE.json config 0/3), P = 5 + 2 n_c n_m doubles:
 *   Mc [s], q, t_c [s], phi_c [rad], 1/D, then T^c_m (re, im) mode-major, channel-minor.
 * t_shift (reading R32): an optional per-walker linear phase term kept OUTSIDE the spline,
 *   Psi_m(f) = spline_m(f) + 2 pi f t_shift for every mode m; DEV [n_w] seconds, or NULL.  With the node phases given
 *   without their 2 pi f t_c term the spline carries ~1e4 rad instead of ~1e7 at the top of a one-year band.
 */
#ifndef LL_B200_H
#define LL_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ll_ctx ll_ctx; /* opaque; owns every internal device buffer */

enum {
    LL_OK = 0,
    LL_ERR_ARG = -1,         /* null pointer, bad size, non-ascending nodes/edges, nodes not covering the grid */
    LL_ERR_STATE = -2,       /* ll_set_data / ll_het_prepare / ll_standin_config not called yet            */
    LL_ERR_CUDA = -3,        /* a CUDA runtime call failed (text in ll_last_error)                         */
    LL_ERR_NOMEM = -4,       /* device or host allocation failed                                           */
    LL_ERR_UNSUPPORTED = -5, /* n_channels / n_modes / precision outside what is compiled in               */
    LL_ERR_REF_ZERO = -6     /* heterodyne reference h0 is zero or non-finite at a bin edge                */
};

enum { LL_PREC_FP64 = 0, LL_PREC_FP32_ACC = 1 };
enum { LL_BC_NATURAL = 0, LL_BC_NOT_A_KNOT = 1 }; /* not-a-knot needs n_nodes >= 4; ll_tlm_nodes is natural-only */

#define LL_MAX_MODES 8
#define LL_MAX_CHANNELS 3

typedef struct {
    int32_t device;     /* CUDA device ordinal                                                              */
    int32_t n_channels; /* 2 (TDI A, E) or 3 (A, E, T: Eq. 3; reading R5)                   */
    int32_t n_modes;    /* 1..LL_MAX_MODES harmonics (l,m) summed per channel (Eq. 9)                       */
    int32_t precision;  /* LL_PREC_FP64, or LL_PREC_FP32_ACC (full-grid path only; reading R15)             */
    int32_t spline_bc;  /* LL_BC_NATURAL (reading R1) or LL_BC_NOT_A_KNOT: boundary condition of every node spline   */
    int32_t reserved[3];
} ll_config;

/* Create / destroy a context.  ll_create selects `device`, checks it is usable and allocates nothing big. */
int ll_create(const ll_config *cfg, ll_ctx **out);
int ll_destroy(ll_ctx *ctx);
const char *ll_last_error(const ll_ctx *ctx);
/* ABI version of the loaded library (bumped on any signature change). */
int ll_abi_version(void);

/* F0 — fix the data stream and the noise weights (Eq. 3; "prior to the analysis, we transform the data",
 * PAPER.md:91).  Builds g^c_i = W^c_i conj(d^c_i) (interleaved [n_f][n_c][re, im]) and
 * <d|d> = sum_c sum_i W^c_i |d^c_i|^2.  May be called again at any time; invalidates ll_het_prepare and every
 * table cached for the previous grid.
 *   d : DEV [n_c][n_f][2]
 *   W : DEV [n_f] when w_shared != 0 (one PSD for every channel: "A=E identical"), else DEV [n_c][n_f]
 *       (W^c_i = 4 df w_i / S^c_n(f_i): every channel its own PSD, "T different").
 * FP32-accumulate contexts take two channels with w_shared != 0 only (LL_ERR_UNSUPPORTED otherwise).       */
int ll_set_data(ll_ctx *ctx, int64_t n_f, int64_t k_min, double df, const double *d, const double *W, int32_t w_shared,
                void *stream);

/* <d|d> over the whole grid and over the heterodyne band (0 before ll_het_prepare).  HOST out.
 * Synchronises `stream` (the one the producing call ran on).                                              */
int ll_get_dd(ll_ctx *ctx, double *dd_full, double *dd_het_band, void *stream);

/* Stand-in waveform description (reading R9): modes (l,m), relative amplitudes c_lm, taper width kappa.
 *   l, m, c_lm : HOST [n_modes]   (n_modes must equal the context's)                                      */
int ll_standin_config(ll_ctx *ctx, int32_t n_modes, const int32_t *l, const int32_t *m, const double *c_lm,
                      double taper_kappa);
/* on != 0: the stand-in entry points of the full-grid path (ll_full_batch_standin, ll_full_template_standin,
 * ll_standin_nodes, ll_pt_*_full) build the node phases WITHOUT the linear term 2 pi f t_c and carry it as
 * t_shift = t_c outside the spline (reading R32).  Same template up to rounding; off by default (reading R2).   */
int ll_standin_split_tc(ll_ctx *ctx, int32_t on);

/* F2-F4 — full-grid log-likelihood of n_w walkers given node arrays (Eq. 2, 3, 7, 9; spline: reading R1).
 *   f_nodes : HOST [n_nodes] strictly ascending, n_nodes >= 3, f_nodes[0] <= f_0, f_nodes[last] >= f_{n_f-1}
 *   amp, phase : DEV [n_w][n_m][n_nodes]  (phase in radians; h_lm = amp exp(-i phase))
 *   tf   : DEV [n_w][n_m][n_c][2]         transfer factors T^c_lm (Eq. 8-9 as per-walker constants, R5/R11)
 *   band : DEV [n_w][2] (f_lo, f_hi) or NULL (whole grid); template is zero outside (reading R10)
 *   t_shift : DEV [n_w] or NULL (see the top of this file; reading R32)
 *   logL, d_h, h_h : DEV [n_w]; d_h and/or h_h may be NULL.  n_w = 0 is a no-op.                          */
int ll_full_batch(ll_ctx *ctx, int64_t n_w, int32_t n_nodes, const double *f_nodes, const double *amp,
                  const double *phase, const double *tf, const double *band, const double *t_shift, double *logL,
                  double *d_h, double *h_h, void *stream);

/* F2-F4 with a frequency-dependent transfer function — h^c(f) = sum_lm T^c_lm(f, t_lm(f)) h_lm(f) (Eq. 8-9,
 * PAPER.md:100-110).  The transfer function's formula is in the paper's ref. [44], so T arrives at the nodes:
 *   tf_nodes : DEV [n_w][n_m][n_c][n_nodes][2]  (re, im); Re T and Im T are splined exactly like amp and phase
 *              (natural cubic in f) and evaluated at every dense bin.  Other arguments as ll_full_batch.
 * FP64 contexts only (LL_ERR_UNSUPPORTED otherwise).                                                        */
int ll_full_batch_tf(ll_ctx *ctx, int64_t n_w, int32_t n_nodes, const double *f_nodes, const double *amp,
                     const double *phase, const double *tf_nodes, const double *band, const double *t_shift, double *logL,
                     double *d_h, double *h_h, void *stream);

/* F2-F4 with PER-WALKER node grids: every walker brings its own nodes, spanning its own band,
 * so each walker has its own tridiagonal system (a true batched solve) and its own bin -> interval map.
 *   f_nodes_w : DEV [n_w][n_nodes], strictly ascending per walker (not checked: the array lives on the device)
 *   amp, phase, tf, band, outputs: as ll_full_batch.  A spline is not extrapolated: the template of walker w is
 *   zero outside [f_nodes_w[w][0], f_nodes_w[w][n_nodes-1]] (intersected with `band` when given; reading R30).
 * FP64 contexts only.                                                                                        */
int ll_full_batch_pw(ll_ctx *ctx, int64_t n_w, int32_t n_nodes, const double *f_nodes_w, const double *amp,
                     const double *phase, const double *tf, const double *band, const double *t_shift, double *logL,
                     double *d_h, double *h_h, void *stream);

/* F1 utility — the stand-in's node arrays in the caller layout (what ll_full_batch_standin builds internally):
 *   params : DEV [n_w][P];  amp, phase : DEV out [n_w][n_m][n_nodes] (phase in radians);
 *   band   : DEV out [n_w][2] = (f_0, min(f_last, (1+kappa) f_ISCO max_m(m/2))) (reading R10), or NULL.
 * Needs ll_standin_config and ll_set_data first.                                                            */
int ll_standin_nodes(ll_ctx *ctx, int64_t n_w, int32_t n_nodes, const double *f_nodes, const double *params,
                     double *amp, double *phase, double *band, void *stream);

/* Eq. 8 utility — t_lm(f_j) = t_ref - (1/2pi) dphi_lm/df at the nodes, dphi/df being the first derivative of the
 * natural cubic spline of the node phases (what a caller needs to evaluate T(f, t_lm(f)) at the nodes).
 *   phase : DEV [n_w][n_m][n_nodes] radians;  t_lm : DEV out, same shape, seconds.  Needs ll_set_data first.   */
int ll_tlm_nodes(ll_ctx *ctx, int64_t n_w, int32_t n_nodes, const double *f_nodes, const double *phase,
                 double t_ref, double *t_lm, void *stream);

/* F1-F4 — same, the node arrays produced on the device from parameter rows by the stand-in waveform.
 *   params : DEV [n_w][P]                                                                                 */
int ll_full_batch_standin(ll_ctx *ctx, int64_t n_w, int32_t n_nodes, const double *f_nodes,
                          const double *params, double *logL, double *d_h, double *h_h, void *stream);

/* End-to-end form of the call above: PINNED (or pageable) HOST params in, HOST results out; the H2D and D2H
 * copies run on `stream`, which is synchronised before returning.                                         */
int ll_full_batch_standin_host(ll_ctx *ctx, int64_t n_w, int32_t n_nodes, const double *f_nodes,
                               const double *params_host, double *logL_host, double *d_h_host,
                               double *h_h_host, void *stream);

/* Dense template of ONE walker through the spline path (what F3 integrates, written out; setup utility
 * used to synthesise data d = h_inj + n).   params_row : HOST [P]   h_out : DEV [n_c][n_f][2]             */
int ll_full_template_standin(ll_ctx *ctx, int32_t n_nodes, const double *f_nodes, const double *params_row,
                             double *h_out, void *stream);

/* Stand-in template of ONE parameter row evaluated directly (no spline) at arbitrary frequencies; zero
 * outside [f_lo, f_hi].  Used for the heterodyne reference h0 (reading R12).
 *   params_row : HOST [P]   f : DEV [n_freq]   h_out : DEV [n_c][n_freq][2]                               */
int ll_template_standin(ll_ctx *ctx, const double *params_row, int64_t n_freq, const double *f, double f_lo,
                        double f_hi, double *h_out, void *stream);

/* H0 — heterodyne summary data for reference template h0 on bins [e_b, e_{b+1}) (last closed), centre
 * f_b = (e_b+e_{b+1})/2 (Eq. 15, 16, 18, 19 with 4 Delta f folded into W; readings R11-R13), 1/h0 at the
 * edges, and <d|d> over the band.  Synchronises `stream` once (it validates h0 at the edges on the host).
 *   f_edges : HOST [n_edges] strictly ascending, n_edges >= 2
 *   h0_dense : DEV [n_c][n_f][2] on the ll_set_data grid      h0_edges : DEV [n_c][n_edges][2]            */
int ll_het_prepare(ll_ctx *ctx, int32_t n_edges, const double *f_edges, const double *h0_dense,
                   const double *h0_edges, void *stream);

/* H0 inside the sampling loop — "The reference template is updated every 5000 iterations of the sampler by
 * replacing it with the highest Likelihood point in the population"; the band is where h0 != 0
 * (PAPER.md:204-210).  Picks the walker with the largest finite log L (lowest index on ties), evaluates its
 * stand-in template directly on the dense grid and at n_edges log-spaced edges
 * f_edges = geomspace(f_0, min(f_{n_f-1}, f_ISCO(best)), n_edges) (reading R12) on the device, and runs H0 on
 * them (everything ll_het_prepare does).  Synchronises `stream`.
 *   params : DEV [n_w][P]   logL : DEV [n_w]   best_index : HOST out (may be NULL)
 *   f_edges_out : HOST out [n_edges] (may be NULL).
 * LL_ERR_ARG when no log L is finite; LL_ERR_REF_ZERO when the best walker's f_ISCO lies below the grid.     */
int ll_het_refresh_standin(ll_ctx *ctx, int64_t n_w, const double *params, const double *logL, int32_t n_edges,
                           int64_t *best_index, double *f_edges_out, void *stream);

/* Audit — "the brute-force Likelihood can ... verify the Heterodyning results": log L, <d|h>, <h|h>
 * of each walker summed bin by bin over the dense bins the heterodyne bins cover (three-term form, Eq. 2-3, with
 * <d|d> over the same bins), the stand-in template evaluated directly at every bin — no spline, no heterodyne.
 * Compare with ll_het_batch_standin on the same rows.   params : DEV [n_w][P]; outputs as ll_het_batch.      */
int ll_het_audit_standin(ll_ctx *ctx, int64_t n_w, const double *params, double *logL, double *d_h, double *h_h,
                         void *stream);

/* Summary data as computed by ll_het_prepare, for inspection.  HOST out, any pointer may be NULL.
 *   A0, A1 : [n_c][n_b][2]    B0, B1 : [n_c][n_b]                                                         */
int ll_het_get_summary(ll_ctx *ctx, double *A0, double *A1, double *B0, double *B1, void *stream);

/* H1-H3 — heterodyned log-likelihood given amplitude/phase at the bin edges (Eq. 11, 14, 17).
 *   amp_e, phase_e : DEV [n_w][n_m][n_edges]   tf : DEV [n_w][n_m][n_c][2]   outputs as ll_full_batch
 *   t_shift : DEV [n_w] or NULL: Psi_m(f_e) = phase_e + 2 pi f_e t_shift (reading R32)                    */
int ll_het_batch(ll_ctx *ctx, int64_t n_w, const double *amp_e, const double *phase_e, const double *tf,
                 const double *t_shift, double *logL, double *d_h, double *h_h, void *stream);

/* H1-H3 with the stand-in waveform evaluated at the edges on the device.   params : DEV [n_w][P]          */
int ll_het_batch_standin(ll_ctx *ctx, int64_t n_w, const double *params, double *logL, double *d_h,
                         double *h_h, void *stream);

/* End-to-end form: HOST params in, HOST results out, copies on `stream`, synchronised before returning.   */
int ll_het_batch_standin_host(ll_ctx *ctx, int64_t n_w, const double *params_host, double *logL_host,
                              double *d_h_host, double *h_h_host, void *stream);

/* ---- Sampler step around the likelihood ------------------------------------------------
 * "This sampler is based on the overall structure of emcee with the parallel tempering scheme from ptemcee ...
 * the typical 'stretch' proposal".  The formulas are in the paper's refs [72]-[74]; readings
 * R25-R28.  The random numbers are INPUTS (uniform on [0,1)), so a step is a deterministic function.
 * A position is a stand-in parameter row [P]; temperatures and walkers are laid out [n_temps][n_walkers].
 *
 * ll_pt_stretch_half_*: update half `half` (0: walkers [0, n/2); 1: [n/2, n)) of every temperature in place.
 *   Walker k draws partner j = floor(u_partner n/2) from the other half and z = ((a-1) u_z + 1)^2 / a;
 *   Y = X_j + z (X_k - X_j); accepted when ln u_accept < (n_dim-1) ln z + beta_t (ln L(Y) - ln L(X_k)), Y inside
 *   [lo, hi] (uniform priors, Table I) and ln L(Y) finite.  ln L(Y) comes from the heterodyned (_het) or the
 *   full-grid (_full) stand-in path of this context: three launches (propose, likelihood, accept), no host sync.
 *   x : DEV [n_temps][n_walkers][P] in/out    logL : DEV [n_temps][n_walkers] in/out (must hold ln L(x) on entry)
 *   d_h, h_h : DEV, same shape, in/out, or NULL    betas : DEV [n_temps]    lo, hi : DEV [P] (+-inf allowed)
 *   n_dim : number of sampled (non-frozen) coordinates    a : stretch scale (2)
 *   u_z, u_partner, u_accept : DEV [n_temps][n_walkers/2]    accepted : DEV out [n_temps][n_walkers/2] or NULL
 * ll_pt_swap: for t = n_temps-1 .. 1, walker i of temperature t and walker i of t-1 exchange (x, ln L, d_h, h_h)
 *   when ln u_swap[t-1][i] < (beta_t - beta_{t-1}) (ln L_{t-1,i} - ln L_{t,i}).   u_swap : DEV [n_temps-1][n_walkers]
 * ll_pt_stats: out3 (DEV [3]) = max finite ln L, its index (as a double; lowest on ties, -1 if none), max
 *   extracted SNR <d|h>/sqrt(<h|h>) — what the two stopping tests look at.
 * ll_stop_snr / ll_stop_converged: the stopping functions themselves (host): 1 = stop. */
int ll_pt_stretch_half_het(ll_ctx *ctx, int32_t n_temps, int32_t n_walkers, int32_t half, double *x, double *logL,
                           double *d_h, double *h_h, const double *betas, const double *lo, const double *hi,
                           int32_t n_dim, double a, const double *u_z, const double *u_partner, const double *u_accept,
                           int32_t *accepted, void *stream);
/* ll_pt_stretch_half_het_static: ll_pt_stretch_half_het for callers that must not allocate (a caller under CUDA
 *   graph capture, a tight serving loop, a harness that forbids cudaMalloc).  Same arguments, same three launches
 *   (propose, H1-H3, accept), same arithmetic (readings R25-R28), results identical to
 *   ll_pt_stretch_half_het; but the step's scratch — the proposal rows [n_temps n_walkers/2][P], their ln L, <d|h>,
 *   <h|h>, (n_dim-1) ln z and inside-the-box flags — lives in a file-scope device array of the library instead of the
 *   context's lazily grown buffers, so this call makes no cudaMalloc, cudaFree or allocating library call, on the
 *   first call or any later one.  ll_het_prepare and ll_standin_config (which do allocate) come before, as for
 *   ll_pt_stretch_half_het.  The array is LL_STATIC_SCRATCH_BYTES (2 MiB) on every GPU that loads the library, held
 *   until the process exits; its device address is looked up once per device in ll_create (cudaGetSymbolAddress with
 *   that device current).
 *   Limit: n_temps (n_walkers/2) (P + 4.5) doubles <= LL_STATIC_SCRATCH_BYTES / 8, e.g. 19 418 proposals at P = 9
 *   (Module-2 size, 10 x 400, needs 2000); beyond it the call returns LL_ERR_ARG, launches nothing, and
 *   ll_last_error names the size asked for and the limit.
 *   ONE array per device, shared by every context and every call: calls that overlap on the GPU (different streams,
 *   different contexts on one device) race on it — serialise them (one stream, or events).  It keeps the last call's
 *   contents; nothing in it has to be cleared, since every element a call reads it has written before.          */
#define LL_STATIC_SCRATCH_BYTES (2 * 1024 * 1024)
int ll_pt_stretch_half_het_static(ll_ctx *ctx, int32_t n_temps, int32_t n_walkers, int32_t half, double *x,
                                  double *logL, double *d_h, double *h_h, const double *betas, const double *lo,
                                  const double *hi, int32_t n_dim, double a, const double *u_z,
                                  const double *u_partner, const double *u_accept, int32_t *accepted, void *stream);
int ll_pt_stretch_half_full(ll_ctx *ctx, int32_t n_nodes, const double *f_nodes, int32_t n_temps, int32_t n_walkers,
                            int32_t half, double *x, double *logL, double *d_h, double *h_h, const double *betas,
                            const double *lo, const double *hi, int32_t n_dim, double a, const double *u_z,
                            const double *u_partner, const double *u_accept, int32_t *accepted, void *stream);
int ll_pt_swap(ll_ctx *ctx, int32_t n_temps, int32_t n_walkers, double *x, double *logL, double *d_h, double *h_h,
               const double *betas, const double *u_swap, int32_t *swapped, void *stream);
int ll_pt_stats(ll_ctx *ctx, int64_t n, const double *logL, const double *d_h, const double *h_h, double *out3,
                void *stream);
/* ll_pt_run_*: n_iter whole iterations (half 0, half 1, swap sweep; iterations iter0 .. iter0 + n_iter - 1) with the
 *   library's own counter-based uniforms (reading R31: SplitMix64; u[kind][index] of iteration it is
 *   mix(mix(seed + G (8 it + kind + 1)) + G (index + 1)) >> 11, times 2^-53; kinds 0-2 = u_z, u_partner, u_accept of
 *   half 0, 3-5 of half 1, 6 = u_swap; G = 0x9E3779B97F4A7C15), so a run is a pure function of (seed, iter0, state).
 *   Everything is enqueued on `stream` (9 launches per iteration for the heterodyned likelihood) and nothing returns to
 *   the host in between; call ll_pt_stats and the stopping functions between runs (every 150 iterations in the paper).
 *   n_accepted : DEV [n_temps] uint64, accepted proposals are ADDED to it (zero it first), or NULL.            */
int ll_pt_run_het(ll_ctx *ctx, int32_t n_temps, int32_t n_walkers, double *x, double *logL, double *d_h, double *h_h,
                  const double *betas, const double *lo, const double *hi, int32_t n_dim, double a, uint64_t seed,
                  int64_t iter0, int64_t n_iter, uint64_t *n_accepted, void *stream);
int ll_pt_run_full(ll_ctx *ctx, int32_t n_nodes, const double *f_nodes, int32_t n_temps, int32_t n_walkers, double *x,
                   double *logL, double *d_h, double *h_h, const double *betas, const double *lo, const double *hi,
                   int32_t n_dim, double a, uint64_t seed, int64_t iter0, int64_t n_iter, uint64_t *n_accepted, void *stream);
/* ll_pt_run_het runs the WHOLE loop as one cooperative launch (a grid of one block per SM that keeps the summary table
 * in shared memory and separates the half updates and the swap sweep by grid barriers) when the context has one mode,
 * n_temps <= 32, and the device supports cooperative launches; otherwise — and always after ll_pt_fused(ctx, 0) — it
 * enqueues 9 launches per iteration.  Both forms are the same function of (seed, iter0, state): same uniforms, same
 * arithmetic, same decisions.                                                                                        */
int ll_pt_fused(ll_ctx *ctx, int32_t on);
typedef struct {
    int32_t n_checks; /* consecutive unchanged checks needed to stop (30 in the paper)   */
    int32_t count;    /* consecutive unchanged checks so far                             */
    int32_t has_ref;  /* 0 before the first check                                        */
    int32_t reserved;
    double tol;       /* "does not change its value by 1": 1.0                           */
    double ref;       /* the value the current run of unchanged checks started from      */
} ll_stop_state;
int ll_stop_snr(double extracted_snr, double limit);
int ll_stop_converged(ll_stop_state *s, double max_logL);

/* Memory check (no part of the method): every internal device buffer has a canary-filled guard band behind it;
 * this synchronises the device, reads the bands back and returns in *n_bad the number of buffers whose band was
 * written (an out-of-bounds store by a kernel; ll_last_error names them).  HOST out.                          */
int ll_debug_check(ll_ctx *ctx, int32_t *n_bad);

/* Measurement helpers (no part of the method).
 * ll_peak_fma: runs `iters` dependent-free FMA chains on every SM and returns the achieved rate in
 *   FMA/s (HOST out); which = 0 -> FP64 DFMA (two loop-invariant register operands), 1 -> FP32 FFMA,
 *   2 -> DFMA with three distinct register operands, 3 -> DFMA with one constant-bank operand,
 *   4 / 5 -> pattern 3 plus 1 integer add per 2 / per 1 DFMA, 6 / 7 -> pattern 3 plus 1 FFMA per 2 / per 1 DFMA
 *   (the rate returned always counts the DFMAs only).
 *   Used for the ALU roofline denominator and for the operand-pattern note under profiles/.
 * ll_kernel_launches: number of kernels this context has launched since creation.
 * ll_last_full_stats: HOST out, after the stream is idle: active (walker, bin, mode) pairs and number of
 *   frequency tiles x walker blocks of the last full-grid call.                                           */
int ll_peak_fma(ll_ctx *ctx, int32_t which, int64_t iters, double *fma_per_s, double *ms, void *stream);
/* ll_profile_enable(on): while on, every full-grid call brackets its fused kernel (F3) and every heterodyned call
 *   its batch kernel (H1-H3) with CUDA events on the call's stream (a ring of 512 pairs; enabling resets it).
 * ll_profile_read: synchronises the recorded events and returns the summed device time in ms and the number
 *   of bracketed launches since the last enable.  HOST out.                                                */
int ll_profile_enable(ll_ctx *ctx, int32_t on);
int ll_profile_read(ll_ctx *ctx, double *kernel_ms_sum, int64_t *n_launches);
int64_t ll_kernel_launches(const ll_ctx *ctx);
int ll_last_full_stats(ll_ctx *ctx, double *active_pairs, int64_t *n_blocks, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* LL_B200_H */
