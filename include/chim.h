/*
 * chim.h -- C ABI of libchim: the B200-native hot path of the CHIMERA-2.0 hierarchical likelihood
 * (arXiv:2504.02034; citations are /root/reference PAPER.md:<line>, readings R1.., M1.. are in DESIGN.md).
 *
 * What one chim_loglike_batch call computes, for every hyper-parameter point lambda in the batch:
 *
 *   log L(lambda) = sum_i log I_i(lambda) - N_events * log xi(lambda)             (eq. 3)
 *
 *   I_i  = int dz  K_gw,i(z | lambda) * p_gal,i(z) [* psi/J on the grid if placement = ON_GRID]
 *          (eq. 14, N_pix = 1), evaluated as a composite trapezoid on event i's own
 *          redshift grid, with K_gw,i the weighted Gaussian KDE of the event's posterior samples in
 *          redshift ("single-1d" kernel, eq. 19):
 *              K_i(z) = 1/(N_s h sqrt(2 pi)) sum_j w_j exp(-(z - z_j)^2 / (2 h^2))
 *          z_j solves d_L^gw(z_j; lambda) = d_L,j with d_L^gw = Xi(z) d_L^em(z), Xi = Xi0 + (1-Xi0)/(1+z)^n
 *          (PAPER.md:17 eq. 1, :23 eq. 2, :52); m_{1,2} = m^d_{1,2}/(1+z_j);
 *              w_j = p(m1,m2 | lambda_m) * [psi(z_j)/((1+z_j)^3 |d d_L^gw/dz|)]^{ON_SAMPLES} / pi_j
 *          (PAPER.md:112 eq. 16 weights, :75 eq. 11 Jacobian, :195 eq. 20 mass model, :226 eq. 21 rate).
 *   xi   = (1/N_inj) sum_{j in detected} s_j,   s_j = p_pop^d(theta_j | lambda) / p_draw,j
 *          (eq. 12) with N_eff from PAPER.md:91 eq. 13.
 *
 * lambda is 15 doubles: H0 [km/s/Mpc], Om, Xi0, n, alpha, beta, delta_m, m_low, m_high, mu_g, sigma_g,
 * lambda_g, gamma, kappa, z_p  (Table 1).
 *
 * Ownership: the caller owns every pointer it passes.  chim_init_* copy and re-pack their inputs before
 * returning (inputs may be freed at once).  Outputs are caller-allocated.  The context owns its device
 * memory until chim_destroy.  Calling an init again replaces the previous set.
 *
 * Threads/streams: one context per stream; calls on one context are not re-entrant.
 *
 * Errors: every int-returning call returns CHIM_OK (0) or a negative chim_status; the message is
 * available from chim_last_error(ctx).  Nothing aborts or throws across the boundary.  Numerical
 * conditions are per-lambda and do not fail the call: they set bits in out_flags (CHIM_FLAG_*).
 *
 * There is no CPU fallback: every entry point that computes needs a CUDA device of compute
 * capability 10.0 (sm_100a).
 */
#ifndef CHIM_H
#define CHIM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CHIM_VERSION 100 /* 0.1.0 */
#define CHIM_N_LAMBDA_PARAMS 15

typedef enum chim_status {
    CHIM_OK = 0,
    CHIM_EINVAL = -1, /* null pointer, bad size, non-increasing grid, m1d < m2d, non-finite input      */
    CHIM_ESTATE = -2, /* chim_loglike_batch before chim_init_events, debug call on a missing set        */
    CHIM_ECUDA = -3,  /* a CUDA runtime call failed (message holds the CUDA error string)               */
    CHIM_ENOMEM = -4  /* host or device allocation failed                                               */
} chim_status;

enum { CHIM_MEM_HOST = 0, CHIM_MEM_DEVICE = 1 };   /* where the pointers given to chim_init_* live     */
enum { CHIM_ON_SAMPLES = 0, CHIM_ON_GRID = 1 };    /* placement of psi/J (R1): N = per-sample weights  */
enum { CHIM_BW_SCOTT = 0, CHIM_BW_FIXED = 1 };     /* KDE bandwidth rule (R3)                          */
enum { CHIM_KDE_AUTO = 0, CHIM_KDE_DIRECT = 1, CHIM_KDE_POWER = 2, CHIM_KDE_NONE = 3 };
                                                   /* KDE formulation.  AUTO: on equally spaced grids
                                                      the local-expansion form, else (or where it does not fit) the power
                                                      form, else the direct form; DIRECT: one MUFU.EX2 per pair on every
                                                      grid; POWER: as AUTO without the local-expansion form; NONE
                                                      (diagnostic): S3/S4 skipped, I_i = mean sample weight, i.e. the
                                                      integral against a flat p_gal = 1 on an unbounded grid -- times
                                                      S2 alone and serves as a closed-form check                          */

enum { CHIM_KERNEL_GAUSS = 0, CHIM_KERNEL_EPANECHNIKOV = 1 };
                                                   /* KDE kernel shape.  EPANECHNIKOV: K(u) = 3/4 (1 - u^2) on |u| <= 1 with
                                                      u = (z - z_j)/h_E, h_E = sqrt(5) h: the same standard deviation h (and
                                                      bandwidth rule) as the Gaussian kernel.  Exact on any grid through
                                                      prefix sums of q_g, q_g z_g, q_g z_g^2 (no pair loop, no cut-off);
                                                      kde_method and kde_cutoff are ignored; needs placement ON_SAMPLES     */

/* per-lambda flag bits written to out_flags */
#define CHIM_FLAG_LAMBDA_DOMAIN 1u   /* H0<=0, Om not in (0,1], Xi0<=0, delta_m<=0, sigma_g<=0, lambda_g not in
                                        [0,1], m_low<=0, m_high<=m_low, z_p<=-1, non-finite -> loglike = NaN    */
#define CHIM_FLAG_DL_NONMONOTONE 2u  /* d d_L^gw/dz <= 0 at a table node (R16) -> loglike = NaN                  */
#define CHIM_FLAG_EVENT_ZERO 4u      /* some I_i = 0 (all weights zero) -> loglike = -inf                        */
#define CHIM_FLAG_XI_ZERO 8u         /* xi = 0 -> loglike = NaN                                                  */
#define CHIM_FLAG_NEFF_LOW 16u       /* N_eff < neff_factor * N_events (R8); loglike is left untouched           */
#define CHIM_FLAG_TABLE_RANGE 32u    /* a sample's d_L exceeds d_L^gw(z_table_max): that sample gets weight 0    */
#define CHIM_FLAG_BW_DEGENERATE 64u  /* Scott bandwidth undefined (fewer than two samples with non-zero weight, or all at one
                                        redshift; R21) -> that log I_i = NaN                                     */

typedef struct chim_ctx chim_ctx; /* opaque; owns all device copies */

typedef struct chim_config {
    int32_t device;      /* CUDA ordinal                                                                      */
    int32_t mem;         /* CHIM_MEM_HOST | CHIM_MEM_DEVICE: where the chim_init_* input pointers live        */
    void *stream;        /* cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = default stream */
    int32_t placement;   /* CHIM_ON_SAMPLES (default, benchmarked) | CHIM_ON_GRID (paper eq. 14 literally)    */
    int32_t bw_rule;     /* CHIM_BW_SCOTT (default) | CHIM_BW_FIXED (uses fixed_bw[] of chim_init_events)      */
    double kde_cutoff;   /* t: sample-grid pairs with |z_g - z_j| > t*h may be skipped (R9); 0 = never skip    */
    double z_cat_max;    /* z_max of PAPER.md:65 eq. 9: support of the selection-term redshift density (R6)    */
    double z_table_max;  /* extent of the d_C(z) table; samples with z > z_table_max get weight 0 (+ flag)     */
    int32_t n_table;     /* panels of the d_C(z) table on [0, z_table_max] (also the monotonicity check nodes) */
    int32_t n_dl_table;  /* intervals of the per-lambda z(ln d_L) interpolation tables; 0 = spacing ~0.005 in ln d_L */
    int32_t n_win_table; /* panels of the per-lambda window table of int m^beta S(m) dm (M4)                   */
    int32_t lambda_chunk;/* lambdas processed per internal pass (bounds the per-lambda table memory)           */
    double neff_factor;  /* NEFF_LOW is raised if N_eff < neff_factor * N_events (R8)                          */
    int32_t kde_method;  /* CHIM_KDE_AUTO (default) | CHIM_KDE_DIRECT | CHIM_KDE_POWER | CHIM_KDE_NONE                              */
    int32_t n_mass_table;/* intervals of the per-lambda mass table in ln m1                           */
    int32_t count_pairs; /* 1: the KDE kernel also counts its (sample, grid point) pairs for chim_get_stats (slower)     */
    int32_t kde_kernel;  /* CHIM_KERNEL_GAUSS (default) | CHIM_KERNEL_EPANECHNIKOV (reading R19)        */
    int32_t n_bins;      /* sample binning (reading R23): 0 = off (default, exact); > 0: per (event, lambda)
                            the weighted samples are reduced to n_bins pseudo-samples (equal-width bins on their redshift
                            range; weighted mean z, summed weight) before the KDE; bandwidth and 1/N_s stay those of the
                            original samples.  An approximation, O((bin width/h)^2).  n_bins <= 2048 and <= the largest N_s  */
} chim_config;

/* Fills *cfg with the defaults: device 0, HOST, NULL stream, ON_SAMPLES, SCOTT, kde_cutoff 6.0,
 * z_cat_max 1.5, z_table_max 10, n_table 2048, n_dl_table 0 (auto), n_win_table 512, lambda_chunk 1024,
 * neff_factor 5, kde_method AUTO, n_mass_table 1024, count_pairs 0, kde_kernel GAUSS, n_bins 0. */
void chim_default_config(chim_config *cfg);

/* Creates a context on cfg->device.  cfg == NULL means chim_default_config.  *out is set to NULL on error; the
 * reason is then available from chim_last_error(NULL) (kept per calling thread until the next failed chim_create).
 * Fails with CHIM_ECUDA if the device is not of compute capability 10.x. */
int chim_create(const chim_config *cfg, chim_ctx **out);
void chim_destroy(chim_ctx *ctx);
const char *chim_last_error(const chim_ctx *ctx); /* never NULL; "" if no error yet; ctx == NULL: the last failed chim_create */
int chim_version(void);
/* Hash of the sources this library was compiled from (paper_2504_02034_b200/build.py: source_hash(); "unknown" for a build made
 * by hand).  The Python binding refuses a library whose id differs from the sources beside it: a stale libchim.so must not be
 * tested or benchmarked in place of the checked-out code. */
const char *chim_build_id(void);

/*
 * Events (PE samples, the fixed per-event redshift grid, p_gal on it).
 *   sample_off [n_events+1] : CSR offsets into dL/m1d/m2d/ln_prior (ragged N_s allowed, N_s >= 1)
 *   dL [Mpc] > 0, m1d >= m2d > 0 [Msun, detector frame], ln_prior = ln pi(theta^d_j) (any prior, R10)
 *   grid_off [n_events+1]   : CSR offsets into z_grid/p_gal (N_z >= 2 per event)
 *   z_grid strictly increasing and >= 0 per event (uniform or not, R14); p_gal >= 0
 *   fixed_bw [n_events] or NULL: bandwidth h_i > 0 when cfg.bw_rule == CHIM_BW_FIXED
 * All arrays live where cfg.mem says.  Samples are re-ordered internally (sorted by d_L); every
 * per-sample output of the debug calls is returned in the caller's original order.
 */
int chim_init_events(chim_ctx *ctx, int32_t n_events, const int64_t *sample_off, const double *dL,
                     const double *m1d, const double *m2d, const double *ln_prior,
                     const int64_t *grid_off, const double *z_grid, const double *p_gal,
                     const double *fixed_bw);

/*
 * "many-1d" kernel (eq. 18; the pixel sum of PAPER.md:97 eq. 14; reading R20).  Optional; call after
 * chim_init_events.  The entries given to chim_init_events are then (event, pixel) SUB-events -- the PE samples that fall
 * in pixel k, the pixel's own grid and p_gal -- and physical event g owns the sub-events [group_off[g], group_off[g+1]):
 *     I_g = sum_k F_k I_k,  F_k = exp(ln_factor[k])   (the hyperparameter-independent factor of eq. 18: the 2-d sky
 *                                                      KDE at the pixel centre times the pixel area)
 *     loglike = sum_g log I_g - n_groups * log xi;  NEFF_LOW compares with neff_factor * n_groups
 *   group_off [n_groups+1]: starts at 0, strictly increasing, ends at n_events (HOST or DEVICE per cfg.mem)
 *   ln_factor [n_events]  : finite
 * out_event_logI of chim_loglike_batch stays per sub-event.  A sub-event with I_k = 0 does not raise EVENT_ZERO; a group
 * whose sub-events are all zero does (loglike = -inf).  Sparse pixels (reading R24): a sub-event whose Scott bandwidth is
 * undefined under a lambda (fewer than two samples with non-zero weight) is left out of the sum and raises BW_DEGENERATE; a
 * group with no I_k > 0 of which one was left out gives loglike = NaN.  n_groups == 0 removes the grouping (every sub-event is an
 * event: the single-1d kernel); chim_init_events also removes it.
 */
int chim_set_event_groups(chim_ctx *ctx, int32_t n_groups, const int64_t *group_off, const double *ln_factor);

/*
 * The step before the path (one-off): the catalogue term p_cat of PAPER.md:62 eq. 8 on redshift grids, from galaxy lists,
 * at a fixed cosmology (computed once for the whole inference; only Omega_m matters, H0 cancels; R22).
 * For each of n_los lines of sight (an event, or an event's pixel):
 *     p_cat(z) = (1/sum_g w_g) sum_g w_g N(z; z_gal_g, sigma_gal_g) dVc/dz(z) / Z_g,  Z_g = int N(z; z_gal_g, sigma_gal_g) dVc/dz dz
 *   gal_off  [n_los+1] CSR offsets into z_gal / sigma_gal / w_gal (>= 1 galaxy per line of sight)
 *   z_gal >= 0, sigma_gal > 0, w_gal > 0 or NULL (unit weights)
 *   grid_off [n_los+1] CSR offsets into z_grid / p_cat_out;  z_grid >= 0
 * All pointers live where cfg.mem says (p_cat_out too); synchronous.  The result can be passed to chim_init_events as p_gal
 * (complete catalogue, as in the paper's runs; for an incomplete one see chim_build_pgal).
 */
int chim_build_pcat(chim_ctx *ctx, double omega_m, int32_t n_los, const int64_t *gal_off, const double *z_gal,
                    const double *sigma_gal, const double *w_gal, const int64_t *grid_off, const double *z_grid,
                    double *p_cat_out);

/*
 * The same with the completeness terms (PAPER.md:58 eq. 7, :65 eq. 9, :67 eq. 10; reading R25): per line of sight
 *     p_gal(z) = f_R p_cat(z) + [1 - P_compl(z)] u(z),  u(z) = (dVc/dz)(z) / Vc(z_max) on [0, z_max], 0 beyond,
 *     f_R = int_0^z_max P_compl(z) u(z) dz                       (= (1/Vc(z_max)) int dVc P_compl, eq. 10)
 * i.e. eq. 7 with the homogeneously distributed missing galaxies of eq. 9, (1 - f_R) p_miss = (1 - P_compl) u.
 *   compl_off [n_los+1] CSR offsets into z_compl / p_compl (>= 2 nodes per line of sight)
 *   z_compl strictly increasing and >= 0 per line of sight; 0 <= p_compl <= 1: the completeness P_compl at the nodes,
 *           linear in between, constant beyond the first / last node
 *   z_max > 0: the z_max of eq. 9-10 (use cfg.z_cat_max for consistency with the selection term, R6)
 *   f_R_out [n_los] or NULL
 * Everything else as chim_build_pcat.  P_compl = 1 gives p_cat and f_R = 1; P_compl = 0 gives u(z) and f_R = 0.
 */
int chim_build_pgal(chim_ctx *ctx, double omega_m, double z_max, int32_t n_los, const int64_t *gal_off, const double *z_gal,
                    const double *sigma_gal, const double *w_gal, const int64_t *compl_off, const double *z_compl,
                    const double *p_compl, const int64_t *grid_off, const double *z_grid, double *p_gal_out, double *f_R_out);

/*
 * chim_build_pcat for callers that must not allocate device memory: eq. 8 exactly as chim_build_pcat computes it,
 * but nothing is cudaMalloc'ed, cudaFree'd or copied to the host.
 *
 * Why it exists: chim_build_pcat makes device copies of its inputs and needs one double of scratch per galaxy, all from
 * cudaMalloc, and frees them with cudaFree before it returns.  That is fine at start-up.  It is not possible (a) inside a
 * JAX / PyTorch process whose framework has already reserved nearly all of the GPU's memory for its own pool -- a cudaMalloc
 * from a foreign library then fails although the framework has room -- and (b) it is unwelcome between likelihood batches,
 * because cudaMalloc and cudaFree synchronise the whole device and so stall a batch still running on another stream.  Such a
 * caller hands over DEVICE pointers for every input and the output (here always DEVICE, whatever cfg.mem says), and the per-
 * galaxy scratch lives in a fixed array inside the library's device image.
 *
 * The limit: at most CHIM_PCAT_STATIC_MAX_GALAXIES galaxies in one call, over all lines of sight together (2 MiB of fp64; every
 * GPU on which libchim.so is loaded holds that array until the process exits, used or not).  A larger n_gal_total is rejected
 * with CHIM_EINVAL and a message naming both numbers; split the lines of sight over several calls, or use chim_build_pcat.
 *
 *   n_gal_total = gal_off[n_los], passed by value because the offsets are never read on the host.  The kernel checks every
 *                 line of sight's range against it: a line of sight whose galaxy range is empty, negative or ends beyond
 *                 n_gal_total gets NaN on its whole grid (nothing is written outside the array).
 *   everything else as chim_build_pcat; w_gal may be NULL.  The VALUES are not validated (that would need a copy to the host):
 *   sigma_gal <= 0, a negative redshift etc. come out as NaN / inf instead of CHIM_EINVAL.
 *
 * Enqueue-only on cfg.stream: no host synchronisation, the caller synchronises before reading p_cat_out.
 * One array per GPU, shared by all contexts and calls: calls that may overlap on the GPU (other streams, other contexts, other
 * host threads) race on it and corrupt each other's result; calls on one stream are ordered and safe.  The array keeps the
 * previous call's contents; nothing in it needs to start at zero (each line of sight writes its coefficients before reading
 * them), so it is never cleared.
 * The first call on each device also looks the array's device address up (and may load the kernel image): make it once at
 * start-up, before any stream capture and before the phase in which the process must leave the allocator alone.
 */
#define CHIM_PCAT_STATIC_MAX_GALAXIES 262144
int chim_build_pcat_static(chim_ctx *ctx, double omega_m, int32_t n_los, int64_t n_gal_total, const int64_t *gal_off,
                           const double *z_gal, const double *sigma_gal, const double *w_gal, const int64_t *grid_off,
                           const double *z_grid, double *p_cat_out);

/*
 * Detected injections for the selection term: n_det stored injections out of
 * n_inj_total drawn; ln_pdraw = ln of the draw density in (d_L, m1d, m2d) (R7).  Optional: without
 * injections log xi := 0 and loglike = sum_i log I_i.  n_det == 0 removes a previous set.
 */
int chim_init_injections(chim_ctx *ctx, int64_t n_det, int64_t n_inj_total, const double *dL,
                         const double *m1d, const double *m2d, const double *ln_pdraw);

/*
 * The hot path.  lambda [n_lambda x 15] row-major and all outputs are DEVICE pointers; the call only
 * enqueues work on cfg.stream (no host synchronisation) -- the caller synchronises.
 *   out_loglike    [n_lambda]            required
 *   out_event_logI [n_lambda x n_events] or NULL   (log I_i; -inf if I_i = 0, NaN if lambda invalid)
 *   out_logxi      [n_lambda] or NULL    (0 without injections)
 *   out_neff       [n_lambda] or NULL    (N_eff of eq. 13; NaN without injections)
 *   out_flags      [n_lambda] or NULL    (CHIM_FLAG_* bits)
 */
int chim_loglike_batch(chim_ctx *ctx, int32_t n_lambda, const double *lambda, double *out_loglike,
                       double *out_event_logI, double *out_logxi, double *out_neff, uint32_t *out_flags);

/* Same computation with HOST pointers: copies lambda to the device, runs the path, copies the
 * requested outputs back and synchronises cfg.stream before returning (the end-to-end call). */
int chim_loglike_batch_host(chim_ctx *ctx, int32_t n_lambda, const double *lambda, double *out_loglike,
                            double *out_event_logI, double *out_logxi, double *out_neff,
                            uint32_t *out_flags);

/*
 * Gradient of log L with respect to the 15 hyper-parameters (the paper's stated direction: gradient-based samplers,
 * PAPER.md:132, :175).  Central differences with one Richardson step,
 *     dlogL/dlambda_k = [4 D(h_k/2) - D(h_k)] / 3,  D(h) = [logL(lambda + h e_k) - logL(lambda - h e_k)] / 2h,
 *     h_k = rel_step |lambda_k| (rel_step where lambda_k = 0),
 * evaluated on the device through the batched hot path itself: the 60 displaced points of every lambda are 60 more rows of
 * one chim_loglike_batch (61 n_lambda rows in all).  DEVICE pointers, enqueue-only like chim_loglike_batch.
 *   rel_step in (0, 0.5); 5e-3 .. 2e-2 keeps both the O(h^4) truncation and the fp32 noise of the path (~1e-5 in log L)
 *            below 1e-3 of the gradient's scale
 *   out_loglike [n_lambda]       log L at lambda itself
 *   out_grad    [n_lambda x 15]  row-major; NaN / inf where a displaced point is not finite (the derivative is undefined there)
 *   out_flags   [n_lambda] or NULL: OR of the flags of the 61 rows
 * log L is smooth in lambda except where a sample crosses a support edge (m1 = m_high, z = z_cat_max for an injection).
 */
int chim_loglike_grad_batch(chim_ctx *ctx, int32_t n_lambda, const double *lambda, double rel_step, double *out_loglike,
                            double *out_grad, uint32_t *out_flags);

/* Work counters of the last chim_loglike_batch on this context (valid after the stream is synchronised;
 * the call itself synchronises).  kde_pairs_in_cutoff = (sample, grid point) pairs with |z_g - z_j| <= t*h, the
 * algorithmic work of S3; kde_pairs_evaluated = fp32 FMA lane-operations the KDE phase executed: in the direct and
 * power forms one per executed pair (the bands are padded to whole blocks and to the widest sample of a warp
 * pass), in the local-expansion form the coefficient build plus one polynomial per sample;
 * kde_pairs_dense = sum_i N_s,i N_z,i x n_lambda.  The first two are only counted when cfg.count_pairs = 1. */
typedef struct chim_stats {
    uint64_t kde_pairs_evaluated;
    uint64_t kde_pairs_in_cutoff;
    uint64_t kde_pairs_dense;
    uint64_t sample_evals;    /* (sample, lambda) weight evaluations  */
    uint64_t injection_evals; /* (injection, lambda) weight evaluations */
    uint64_t kernel_launches; /* kernels launched by the last batch call */
} chim_stats;
int chim_get_stats(chim_ctx *ctx, chim_stats *out);

/* Per-kernel device times of the last chim_loglike_batch: when profiling is enabled, CUDA events are recorded on
 * cfg.stream around every kernel launch of the batch (no host synchronisation is added to the batch call);
 * chim_get_kernel_times synchronises the stream and sums the elapsed times per kernel kind.  S1 = table
 * builder and polynomial fits; S2-S4 = the fused sample-weight + KDE + integral step, split into k_events_fast (events_*: the
 * regular units) and k_events (events_general_*: every other unit -- all of them when the configuration is not the default
 * one); S5 = injection reduction; S6 = combine. */
typedef struct chim_kernel_times {
    double tables_ms, events_ms, inject_ms, combine_ms;
    uint32_t tables_launches, events_launches, inject_launches, combine_launches;
    double events_general_ms;
    uint32_t events_general_launches;
    uint32_t events_handed_over; /* (event, lambda) units k_events_fast left to k_events in the LAST lambda chunk of the batch */
} chim_kernel_times;
int chim_set_profiling(chim_ctx *ctx, int32_t enable);
int chim_get_kernel_times(chim_ctx *ctx, chim_kernel_times *out);

/* Plain-ALU peak rates of the device the context lives on, measured by micro-benchmarks (independent dependency
 * chains, 8 CTAs per SM) on cfg.stream; synchronous.  These are the roofline denominators of the path, which is
 * bound by the SMs' arithmetic pipes rather than by HBM or the tensor cores.  All four are in
 * 1e9 lane-instructions per second: MUFU.EX2, FFMA, DFMA, and FFMA2 (packed fp32x2, counted as two). */
typedef struct chim_alu_peaks {
    double ex2_gops, ffma_gops, dfma_gops, ffma2_gops;
    int32_t sm_count, reserved;
} chim_alu_peaks;
int chim_measure_alu_peaks(chim_ctx *ctx, chim_alu_peaks *out);

/* ---- diagnostics: intermediates of the path for ONE lambda (DEVICE pointer to 15 doubles) -------------
 * They run the same device code as the hot path and exist so that each step can be compared with the
 * oracle (tests tier T2).  Outputs are DEVICE pointers; any of them may be NULL.  Synchronous. */

/* Step S1: the per-lambda event table.  For n query distances dL[] (inside the d_L range of the event
 * set) returns z(dL) and the smooth redshift factor of the weights, psi(z)/J(z) (1 if ON_GRID). */
int chim_debug_table_lookup(chim_ctx *ctx, const double *lambda, int64_t n, const double *dL,
                            double *z_out, double *ratio_out);
/* Step S2: per-sample redshift and weight of event `event`, in the caller's sample order [N_s]. */
int chim_debug_event_samples(chim_ctx *ctx, const double *lambda, int32_t event, double *z_out,
                             double *w_out);
/* Steps S2-S4: bandwidth h (1 double), KDE on the event grid K_out [N_z] (no cut-off applied to the
 * returned K if kde_cutoff == 0; otherwise the skipped pairs are missing from it), and log I.
 * K_out is available for the Gaussian kernel only (NaN with CHIM_KERNEL_EPANECHNIKOV). */
int chim_debug_event_kde(chim_ctx *ctx, const double *lambda, int32_t event, double *h_out, double *K_out,
                         double *logI_out);
/* Step S5: per-injection s_j in the caller's order [n_det]. */
int chim_debug_injection_weights(chim_ctx *ctx, const double *lambda, double *s_out);

#ifdef __cplusplus
}
#endif
#endif /* CHIM_H */
